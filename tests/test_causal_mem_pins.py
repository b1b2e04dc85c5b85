"""Pins for oracle/uf_causal_mem.py: each one ties a function of the oracle to something other
than itself — a library routine (torch CPU conv2d / pixel_shuffle in fp64), a brute-force loop written from Eq. 2
(PAPER.md:65), a closed form, or an invariant the paper states (variant A == variant B, causality)."""
import itertools

import numpy as np
import pytest
import torch

import uf_workloads as wl
from oracle import uf_causal_mem as cm


def _cfg(c: wl.CmnWorkload) -> cm.CmnConfig:
    return cm.CmnConfig(c.in_ch, c.out_ch, tuple(c.stage_channels), c.n_blocks, tuple(c.spatial_factors),
                        tuple(c.temporal_factors))


def _wt64(c: wl.CmnWorkload, seed=30_000):
    return {k: v.astype(np.float64) for k, v in wl.cmn_weights(c, seed).items()}


def _frames64(c, chunk, frames=None):
    return wl.bf16_bits_to_f32(wl.cmn_frames(c, chunk, frames)).astype(np.float64)


SMALL = wl.CmnWorkload("pin", 4, 3, (8, 6), 2, (2, 1), (1, 2), 5, 7, 2)


# ---- bf16 rounding -------------------------------------------------------------------------------------------
def test_round_bf16_matches_bit_level_rounding_of_fp32_values():
    g = np.random.default_rng(1)
    x = np.concatenate([g.standard_normal(20000).astype(np.float32) * np.float32(10.0) ** g.integers(-30, 30, 20000),
                        np.array([0.0, -0.0, 1.0, 1.00390625, 1.01171875, 3.3895314e38, 1e-40, -1e-45], np.float32)])
    ref = wl.bf16_bits_to_f32(wl.f32_to_bf16_bits(x)).astype(np.float64)       # integer add-and-shift on the bits
    got = cm.round_bf16(x.astype(np.float64))
    assert np.array_equal(got, ref)


def test_round_bf16_rounds_fp64_once_and_ties_to_even():
    # 1 + 2^-8 is halfway between the bf16 numbers 1 and 1 + 2^-7: even mantissa wins (1.0); 1 + 3*2^-8 -> 1 + 2^-6
    assert cm.round_bf16(np.array([1 + 2.0 ** -8]))[0] == 1.0
    assert cm.round_bf16(np.array([1 + 3 * 2.0 ** -8]))[0] == 1 + 2.0 ** -6
    # just above the tie in fp64 (invisible after a first rounding to fp32) must round up: single rounding
    assert cm.round_bf16(np.array([1 + 2.0 ** -8 + 2.0 ** -40]))[0] == 1 + 2.0 ** -7
    assert cm.round_bf16(np.array([-(1 + 2.0 ** -8 + 2.0 ** -40)]))[0] == -(1 + 2.0 ** -7)
    # any memory layout (a transposed view once came back as uninitialised memory)
    g = np.random.default_rng(11)
    a = g.standard_normal((3, 4, 5))
    assert np.array_equal(cm.round_bf16(a.transpose(2, 0, 1)), cm.round_bf16(a).transpose(2, 0, 1))
    assert np.array_equal(cm.round_bf16(np.asfortranarray(a)), cm.round_bf16(a))


# ---- conv3x3 / conv1x1 against the library routine and special cases -------------------------------------------
def test_conv3x3_equals_torch_conv2d_fp64():
    g = np.random.default_rng(2)
    x = g.standard_normal((2, 6, 9, 5))
    w = g.standard_normal((7, 5, 3, 3))
    b = g.standard_normal(7)
    ref = torch.nn.functional.conv2d(torch.from_numpy(x).permute(0, 3, 1, 2), torch.from_numpy(w), torch.from_numpy(b),
                                     padding=1).permute(0, 2, 3, 1).numpy()
    assert np.allclose(cm.conv3x3(x, w, b), ref, rtol=0, atol=1e-12)


def test_conv3x3_identity_kernel_and_delta_input():
    g = np.random.default_rng(3)
    x = g.standard_normal((1, 5, 6, 4))
    w = np.zeros((4, 4, 3, 3))
    w[np.arange(4), np.arange(4), 1, 1] = 1.0
    assert np.array_equal(cm.conv3x3(x, w, None), x)
    # a unit impulse at (2,3) in channel 1 spreads the FLIPPED kernel around it (cross-correlation, R-42):
    # out[y,x,o] = w[o,1,2-y+1... ] i.e. out[2-dy+1, 3-dx+1, o] = w[o,1,dy,dx]
    w = g.standard_normal((3, 4, 3, 3))
    d = np.zeros((1, 5, 6, 4))
    d[0, 2, 3, 1] = 1.0
    out = cm.conv3x3(d, w, None)
    for dy, dx, o in itertools.product(range(3), range(3), range(3)):
        assert out[0, 2 - (dy - 1), 3 - (dx - 1), o] == w[o, 1, dy, dx]
    assert np.count_nonzero(out) == 27
    # zero padding: an impulse in the corner loses the taps that fall outside
    d = np.zeros((1, 5, 6, 4))
    d[0, 0, 0, 0] = 1.0
    assert np.count_nonzero(cm.conv3x3(d, np.ones((1, 4, 3, 3)), None)) == 4


def test_conv1x1_is_a_per_pixel_matrix_product():
    g = np.random.default_rng(4)
    x = g.standard_normal((2, 3, 4, 5))
    w = g.standard_normal((6, 5))
    b = g.standard_normal(6)
    out = cm.conv1x1(x, w, b)
    for f, y, xx in itertools.product(range(2), range(3), range(4)):
        assert np.allclose(out[f, y, xx], w @ x[f, y, xx] + b, atol=1e-13)


# ---- PixelShuffle / channel-to-time (R-44) --------------------------------------------------------------------
@pytest.mark.parametrize("r", [2, 3])
def test_pixel_shuffle_equals_torch_and_index_formula(r):
    g = np.random.default_rng(5)
    x = g.standard_normal((2, 3, 4, 5 * r * r))
    ref = torch.nn.functional.pixel_shuffle(torch.from_numpy(x).permute(0, 3, 1, 2), r).permute(0, 2, 3, 1).numpy()
    got = cm.pixel_shuffle(x, r)
    assert np.array_equal(got, ref)
    for y, xx, c, i, j in itertools.product(range(3), range(4), range(5), range(r), range(r)):
        assert got[1, y * r + i, xx * r + j, c] == x[1, y, xx, c * r * r + i * r + j]


def test_channel_to_time_index_formula():
    g = np.random.default_rng(6)
    x = g.standard_normal((3, 2, 2, 8))
    got = cm.channel_to_time(x, 2)
    assert got.shape == (6, 2, 2, 4)
    for f, k, c in itertools.product(range(3), range(2), range(4)):
        assert np.array_equal(got[f * 2 + k, :, :, c], x[f, :, :, k * 4 + c])


# ---- the block: brute force from Eq. 2 -------------------------------------------------------------------------
def test_mem_block_equals_per_pixel_loops_of_eq2():
    g = np.random.default_rng(7)
    C, H, W = 3, 4, 5
    rb = cm.round_bf16
    h = rb(g.standard_normal((1, H, W, C)))
    m = rb(g.standard_normal((1, H, W, C)))
    wt = {"c1": rb(g.standard_normal((C, 2 * C, 3, 3)) * 0.3), "c1.b": g.standard_normal(C) * 0.1,
          "c2": rb(g.standard_normal((C, C, 3, 3)) * 0.3), "c2.b": g.standard_normal(C) * 0.1,
          "c3": rb(g.standard_normal((C, C, 3, 3)) * 0.3), "c3.b": g.standard_normal(C) * 0.1,
          "skip": rb(g.standard_normal((C, C)) * 0.3)}

    def conv_px(src, w, b, y, x, o):                 # one output element from the definition, python floats
        acc = 0.0
        for i in range(src.shape[-1]):
            for dy in range(3):
                for dx in range(3):
                    yy, xx = y + dy - 1, x + dx - 1
                    if 0 <= yy < H and 0 <= xx < W:
                        acc += w[o, i, dy, dx] * src[0, yy, xx, i]
        return acc + b[o]

    cat = np.concatenate([h, m], axis=-1)
    a1 = np.zeros((1, H, W, C))
    a2 = np.zeros((1, H, W, C))
    out = np.zeros((1, H, W, C))
    for y, x, o in itertools.product(range(H), range(W), range(C)):
        a1[0, y, x, o] = max(conv_px(cat, wt["c1"], wt["c1.b"], y, x, o), 0.0)
    a1 = rb(a1)
    for y, x, o in itertools.product(range(H), range(W), range(C)):
        a2[0, y, x, o] = conv_px(a1, wt["c2"], wt["c2.b"], y, x, o)
    a2 = rb(a2)
    for y, x, o in itertools.product(range(H), range(W), range(C)):
        skip = sum(wt["skip"][o, i] * h[0, y, x, i] for i in range(C))
        out[0, y, x, o] = max(conv_px(a2, wt["c3"], wt["c3.b"], y, x, o) + skip, 0.0)
    out = rb(out)
    got = cm.mem_block(h, m, {"p." + k: v for k, v in wt.items()}, "p.")
    # the two summation orders differ by fp64 rounding only; a bf16 flip needs a sum within 1e-13 of a tie
    assert np.allclose(got, out, rtol=0, atol=1e-12)


def test_block_with_zero_weights_on_memory_ignores_memory_and_zero_c3_gives_relu_of_skip():
    g = np.random.default_rng(8)
    c = SMALL
    cfg, wt = _cfg(c), _wt64(c)
    h = cm.round_bf16(g.standard_normal((1, 4, 4, 8)))
    m1 = cm.round_bf16(g.standard_normal((1, 4, 4, 8)))
    w2 = dict(wt)
    w2["s0.b0.c1"] = wt["s0.b0.c1"].copy()
    w2["s0.b0.c1"][:, 8:] = 0.0                                   # memory half of the concatenation
    assert np.array_equal(cm.mem_block(h, m1, w2, "s0.b0."), cm.mem_block(h, np.zeros_like(h), w2, "s0.b0."))
    w3 = dict(wt)
    w3["s0.b0.c3"] = np.zeros_like(wt["s0.b0.c3"])
    w3["s0.b0.c3.b"] = np.zeros_like(wt["s0.b0.c3.b"])
    ref = cm.round_bf16(np.maximum(h @ wt["s0.b0.skip"].T, 0.0))
    assert np.array_equal(cm.mem_block(h, m1, w3, "s0.b0."), ref)


# ---- network structure -----------------------------------------------------------------------------------------
def test_parameter_shapes_agree_with_the_generator_and_paper_widths():
    for c in wl.CMN_CONFIGS.values():
        assert cm.weight_names(_cfg(c)) == wl.cmn_param_shapes(c)
    names = dict(cm.weight_names(cm.UPSAMPLER))
    assert names["in"] == (256, 16, 3, 3) and names["s0.b0.c1"] == (256, 512, 3, 3)
    assert names["s0.up"] == (1024, 256, 3, 3) and names["s0.ch"] == (128, 256) and names["s2.ch"] == (64, 64)
    assert names["out"] == (16, 64, 3, 3) and "s0.texp" not in names
    assert len([n for n in names if n.endswith("c1")]) == 9       # 3 blocks x 3 stages
    names = dict(cm.weight_names(cm.HR_DECODER))
    assert names["s1.texp"] == (256, 128) and names["s2.texp"] == (128, 64) and "s0.texp" not in names
    assert names["s2.ch"] == (64, 64) and names["out"] == (3, 64, 3, 3) and names["s2.up"] == (256, 64, 3, 3)


def test_output_shape_and_flop_count_closed_form():
    c = SMALL
    cfg, wt = _cfg(c), _wt64(c)
    out = cm.forward_parallel(_frames64(c, 0, 3), cfg, wt)
    assert out.shape == (3 * 2, 5 * 2, 7 * 2, 3)
    # by hand: px0 = 5*7 per frame; stage 0 at 8 ch, 2 blocks, up 8->32 (r=2), ch 8->6; stage 1 at 6 ch on 4x px,
    # up 6->6, texp 6->12 (frames x2), ch 6->6 on 8x px; out 6->3
    px = 35
    macs = px * (8 * 4 * 9) + 2 * px * (8 * 16 * 9 + 2 * 8 * 8 * 9 + 8 * 8) + px * (32 * 8 * 9) + 4 * px * (6 * 8)
    macs += 2 * 4 * px * (6 * 12 * 9 + 2 * 6 * 6 * 9 + 6 * 6) + 4 * px * (6 * 6 * 9) + 4 * px * (12 * 6) + 8 * px * 36
    macs += 8 * px * (3 * 6 * 9)
    assert cm.flop_count(cfg, 5, 7, 1) == 2 * macs
    assert cm.flop_count(cfg, 5, 7, 3) == 3 * 2 * macs


# ---- variant A == variant B, chunking, causality ------------------------------------------
@pytest.mark.parametrize("name", ["pin", "cmn_tiny"])
def test_streaming_variant_b_equals_parallel_variant_a_frame_by_frame(name):
    c = SMALL if name == "pin" else wl.scaled_cmn(wl.CMN_CONFIGS["cmn_tiny"], height=6, width=9)
    cfg, wt = _cfg(c), _wt64(c)
    T = 5
    z = _frames64(c, 0, T)
    ref = cm.forward_parallel(z, cfg, wt)
    st = cm.CausalMemStream(cfg, wt)
    got = np.concatenate([st.step(z[0:2]), st.step(z[2:3]), st.step(z[3:5])], axis=0)     # chunks of 2, 1, 2 frames
    assert got.shape == ref.shape
    assert np.array_equal(got, ref)
    st.reset()
    again = st.step(z)
    assert np.array_equal(again, ref)


def test_causality_and_memory_dependence():
    c = SMALL
    cfg, wt = _cfg(c), _wt64(c)
    T, s_total = 4, 2
    z = _frames64(c, 0, T)
    ref = cm.forward_parallel(z, cfg, wt)
    z2 = z.copy()
    z2[2] = cm.round_bf16(z2[2] + 1.0)
    alt = cm.forward_parallel(z2, cfg, wt)
    assert np.array_equal(alt[:2 * s_total], ref[:2 * s_total])            # frames before t = 2 unchanged
    assert not np.array_equal(alt[2 * s_total:3 * s_total], ref[2 * s_total:3 * s_total])
    assert not np.array_equal(alt[3 * s_total:], ref[3 * s_total:])        # the next frame sees it through the memory
    # the first frame of a stream sees zero memory: equal to running it alone
    assert np.array_equal(cm.forward_parallel(z[:1], cfg, wt), ref[:s_total])
    # the memory has one frame of reach per block: with a single block per stage, frame t+2 of a one-stage, no-texp
    # net does not see frame t
    c1 = wl.CmnWorkload("reach", 4, 3, (8,), 1, (1,), (1,), 5, 7, 2)
    cfg1, wt1 = _cfg(c1), _wt64(c1)
    za = _frames64(c1, 0, 4)
    zb = za.copy()
    zb[0] = cm.round_bf16(zb[0] + 1.0)
    a, b = cm.forward_parallel(za, cfg1, wt1), cm.forward_parallel(zb, cfg1, wt1)
    assert not np.array_equal(a[1], b[1]) and np.array_equal(a[2:], b[2:])


def test_literal_variant_b_output_memory_differs_from_the_second_frame_on():
    """VERDICT r2 item 8 / ADVICE r2: Alg. 2 variant B as printed stores the block OUTPUT.  With zero initial
    memory the first frame cannot tell the two readings apart; every later frame can.  The output reading is a
    recurrence: frame 0 still reaches frame 3 of a one-block network, where the input reading (one frame of reach per
    block, pinned above) has forgotten it.  Both stay causal."""
    c1 = wl.CmnWorkload("reach", 4, 3, (8,), 1, (1,), (1,), 5, 7, 2)
    cfg, wt = _cfg(c1), _wt64(c1)
    z = _frames64(c1, 0, 4)
    a = cm.CausalMemStream(cfg, wt, memory="input").step(z)
    b = cm.CausalMemStream(cfg, wt, memory="output").step(z)
    assert np.array_equal(a, cm.forward_parallel(z, cfg, wt))
    assert np.array_equal(a[0], b[0])
    for t in (1, 2, 3):
        assert not np.array_equal(a[t], b[t]), t
    # the second frame of the output reading, restated by hand from Eq. 2: memory = the first frame's block output
    h0 = cm.round_bf16(cm.conv3x3(z[0:1], wt["in"], wt["in.b"]))
    h1 = cm.round_bf16(cm.conv3x3(z[1:2], wt["in"], wt["in.b"]))
    out0 = cm.mem_block(h0, np.zeros_like(h0), wt, "s0.b0.")
    out1 = cm.mem_block(h1, out0, wt, "s0.b0.")
    tail = cm.round_bf16(cm.conv3x3(cm._stage_tail(out1, cfg, 0, wt), wt["out"], wt["out.b"]))
    assert np.array_equal(tail[0], b[1])
    # chunking does not matter (state is carried), causality holds, and the reach is unbounded
    st = cm.CausalMemStream(cfg, wt, memory="output")
    assert np.array_equal(np.concatenate([st.step(z[:1]), st.step(z[1:3]), st.step(z[3:])]), b)
    z2 = z.copy()
    z2[0] = cm.round_bf16(z2[0] + 1.0)
    b2 = cm.CausalMemStream(cfg, wt, memory="output").step(z2)
    assert not np.array_equal(b2[3], b[3])                     # frame 0 reaches frame 3 through the recurrence
    z3 = z.copy()
    z3[2] = cm.round_bf16(z3[2] + 1.0)
    b3 = cm.CausalMemStream(cfg, wt, memory="output").step(z3)
    assert np.array_equal(b3[:2], b[:2]) and not np.array_equal(b3[2], b[2])
    # how far apart the two readings are on seeded weights (reported, not asserted beyond "not small")
    rel = np.sqrt(np.mean((a[1:] - b[1:]) ** 2) / np.mean(a[1:] ** 2))
    assert rel > 1e-3, rel
    with pytest.raises(ValueError):
        cm.CausalMemStream(cfg, wt, memory="both")
