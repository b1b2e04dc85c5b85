"""GPU parity of the causal memory network streaming step (NEXT-4, include/uf_cmn.h) against
oracle/uf_causal_mem.py on the same seeded weights and frames: every layer element by element on identical inputs
(one bf16 ulp), network outputs and per-block memories end to end (rounding-noise bound), over streams cut into
ragged chunks; grids that span several CTA tiles with ragged edges; the paper's
two configurations (P:345 upsampler, P:347 decoder) on reduced grids and the upsampler at BASELINE.json's 1K size."""
import numpy as np
import pytest

import uf_workloads as wl
import uf_harness as hz

pytestmark = pytest.mark.gpu


def _run_stream(c, chunks, frames_max=None, layerwise=True, check_memory=True):
    """stream of sum(chunks) frames cut into the given chunk lengths.  Per chunk: (1) every layer of the step against
    the oracle's layer function on the same inputs (one-ulp bound, uf_harness.cmn_layer_check); (2) the network
    output against the oracle's variant A over the whole stream (rounding-noise bound, uf_harness.compare_cmn);
    at the end (3) every block memory against the streaming oracle (variant B)."""
    cm, cfg, wt = hz.cmn_oracle(c)
    T = sum(chunks)
    zb = wl.cmn_frames(c, 0, T)
    z = hz.bits_to_f64(zb)
    ref = cm.forward_parallel(z, cfg, wt)
    cu = hz.CmnCuda(c, frames_max=frames_max or max(chunks))
    ts, nl = cu.ts, cu.uf.uf_cmn_n_layers(cu.net)
    try:
        f0, stats, mem_prev = 0, [], {}
        for i, n in enumerate(chunks):
            got = cu.step(zb[f0:f0 + n])
            st = hz.compare_cmn(got, ref[f0 * ts:(f0 + n) * ts], nl, f"[{c.name} chunk {i}]")
            if layerwise:
                st["layer_min_frac_equal"] = hz.cmn_layerwise(cu, cm, cfg, wt, z[f0:f0 + n], got, mem_prev,
                                                              f"[{c.name} chunk {i}]")
            stats.append(st)
            f0 += n
        if check_memory:
            # memory of every block == the block's input at the last frame (R-41), from the streaming oracle (variant B)
            so = cm.CausalMemStream(cfg, wt)
            so.step(z)
            for s in range(cfg.n_stages):
                for b in range(cfg.n_blocks):
                    hz.compare_cmn(cu.memory(s, b)[None], so.mem[f"s{s}.b{b}."], nl, f"[{c.name} memory s{s}.b{b}]")
        assert cu.uf.uf_cmn_launches(cu.net) == len(chunks) * nl
        assert cu.uf.uf_cmn_flops(cu.net, 1) == cm.flop_count(cfg, c.height, c.width, 1)
        return stats
    finally:
        cu.close()


def test_tiny_network_ragged_chunks_and_memories():
    c = wl.CMN_CONFIGS["cmn_tiny"]                      # 12 x 20 grid: ragged in both directions, r = (2,1), s = (1,2)
    print(_run_stream(c, [2, 1, 2]))


def test_reset_starts_a_new_stream_and_single_frames():
    c = wl.CMN_CONFIGS["cmn_tiny"]
    cm, cfg, wt = hz.cmn_oracle(c)
    zb = wl.cmn_frames(c, 0, 3)
    ref = cm.forward_parallel(hz.bits_to_f64(zb), cfg, wt)
    cu = hz.CmnCuda(c, frames_max=3)
    try:
        a = cu.step(zb)
        cu.reset()
        b = np.concatenate([cu.step(zb[i:i + 1]) for i in range(3)], axis=0)     # frame by frame after a reset
        assert np.array_equal(a, b)
        hz.compare_cmn(a, ref, cu.uf.uf_cmn_n_layers(cu.net), "[reset]")
        # without the reset the first frame sees the previous stream's last frame: a different result
        c2 = cu.step(zb[:1])
        assert not np.array_equal(c2, a[:cu.ts])
    finally:
        cu.close()


def test_multi_tile_grid_with_ragged_edges():
    # 37 x 75: 5 tile rows (last 5 of 8 rows), 2 CTA tiles of 64 columns (MT = 4; last 11 of 64), several frames
    c = wl.scaled_cmn(wl.CMN_CONFIGS["cmn_tiny"], "cmn_ragged", height=37, width=75, frames_per_chunk=3)
    _run_stream(c, [3, 2])


@pytest.mark.parametrize("r", [1, 3])
def test_spatial_factors_1_and_3(r):
    c = wl.CmnWorkload(f"cmn_r{r}", 16, 16, (64,), 1, (r,), (1,), 10, 18, 2)
    _run_stream(c, [2, 2])


def test_wide_channels_n256_and_n128_paths():
    # the upsampler's widths on a small grid: N = 256 tiles with MT = 2, the 1024-column PixelShuffle conv
    # in 4 N tiles, N = 128 with MT = 4, N = 64 double-buffered
    c = wl.scaled_cmn(wl.CMN_CONFIGS["cmn_upsampler_1k"], "cmn_upsampler_small", height=20, width=36, frames_per_chunk=2)
    _run_stream(c, [2, 1])


def test_decoder_configuration_small():
    # spatial (2,2,2), temporal (1,2,2), out_ch = 3 (scalar stores), widths (256,128,64,64)
    c = wl.scaled_cmn(wl.CMN_CONFIGS["cmn_decoder_crop"], "cmn_decoder_small", height=6, width=10, frames_per_chunk=1)
    _run_stream(c, [1, 1])


def test_upsampler_full_1k_chunk():
    # BASELINE.json's 1K grid: LR latent 68 x 120, chunk of 3 latent frames -> 136 x 240 (the launch configuration
    # bench.py times); a second chunk runs on real memories (its first Conv1 of every block is checked layer-wise
    # against the oracle fed with the GPU's own previous frame, so the streaming oracle is not run a third time here)
    c = wl.CMN_CONFIGS["cmn_upsampler_1k"]
    st = _run_stream(c, [3, 1], check_memory=False)
    print("cmn_upsampler_1k parity:", st)


@pytest.mark.parametrize("seed", range(6))
def test_randomised_networks(seed):
    """Seeded random small networks: widths 64 / 128 / 192 / 256 (N = 192 tiles, three 64-channel slices), 1-3 stages,
    spatial factors 1-3, temporal factors 1-3, 1-2 blocks per stage, in_ch 8 / 16 / 24, out_ch 1-40 (GEMM columns padded
    to 16, scalar and vector stores), grids from smaller than one tile to several ragged tiles, ragged chunk lengths."""
    rng = np.random.default_rng(500 + seed)
    n_stages = int(rng.integers(1, 4))
    widths, rs, ts = [], [], []
    for _ in range(n_stages):
        r = int(rng.choice([1, 1, 2, 3]))
        c = int(rng.choice([64, 128, 192, 256] if r == 1 else [64, 128, 256] if r == 2 else [64]))   # C r^2 <= 1024
        widths.append(c); rs.append(r); ts.append(int(rng.choice([1, 1, 2, 3])))
    if rng.random() < 0.5:
        widths.append(int(rng.choice([64, 128])))
    c = wl.CmnWorkload(f"cmn_rand{seed}", int(rng.choice([8, 16, 24])), int(rng.integers(1, 41)), tuple(widths),
                       int(rng.integers(1, 3)), tuple(rs), tuple(ts), int(rng.integers(3, 20)), int(rng.integers(3, 40)), 2)
    chunks = [int(x) for x in rng.integers(1, 4, size=int(rng.integers(1, 4)))]
    print(c, chunks)
    _run_stream(c, chunks, frames_max=3)


def test_decoder_crop_full_size():
    # P:347 on one 68 x 120 latent frame -> 4 frames of 544 x 960 x 3: the second launch configuration bench.py times
    # (64-channel layers on 272 x 480 x 2 frames, N = 64 tiles, 3-channel scalar stores)
    c = wl.CMN_CONFIGS["cmn_decoder_crop"]
    st = _run_stream(c, [1], check_memory=False)
    print("cmn_decoder_crop parity:", st)


def test_decoder_full_1k_sampled_windows():
    """P:347 at the size bench.py times as cmn_decoder_1k: the whole 136 x 240 HR latent, a chunk of 3 latent frames ->
    12 frames of 1088 x 1920 x 3 (the decoder had only been run on a quarter-area, one-frame crop).  The
    tensors are too large for the NumPy oracle as a whole (2.7 TFLOP per frame), so every layer is checked on windows:
    the oracle's layer function on crops of the GPU's own input activations against the GPU's output, within one bf16
    ulp and >= 99 % bit-equal per window (two opposite corners + seeded random frames and positions per layer)."""
    c = wl.CMN_CONFIGS["cmn_decoder_1k"]
    cm, cfg, wt = hz.cmn_oracle(c)
    zb = wl.cmn_frames(c, 0, 3)
    net = hz.CmnCuda(c, frames_max=3)
    try:
        print("cmn_decoder_1k ctx bytes:", net.uf.uf_cmn_device_bytes(net.net))
        out_bits = net.step_bits(zb)
        assert out_bits.shape == (12, 1088, 1920, 3)
        assert np.isfinite(hz.bits_to_f64(out_bits[::4, ::16, ::16])).all()
        eq = hz.cmn_layerwise_sampled(net, cm, cfg, wt, zb, out_bits, n_windows=5, win=20, seed=7, where="[cmn_decoder_1k]")
        print(f"cmn_decoder_1k: every sampled window of every layer within one bf16 ulp, >= {eq:.4f} bit-equal")
    finally:
        net.close()


def test_argument_errors():
    import paper_2606_09150_b200 as uf
    with pytest.raises(uf.UFError) as e:
        uf.uf_cmn_create(16, 16, (48,), 1, (1,), (1,), 8, 8, 1)
    assert e.value.code == uf.binding.UF_ERR_UNSUPPORTED
    c = wl.CMN_CONFIGS["cmn_tiny"]
    net = uf.uf_cmn_create(c.in_ch, c.out_ch, c.stage_channels, c.n_blocks, c.spatial_factors, c.temporal_factors,
                           c.height, c.width, 2, 0)
    try:
        import torch
        z = torch.zeros((2, c.height, c.width, c.in_ch), dtype=torch.bfloat16, device="cuda")
        out = torch.zeros((4, c.height * 2, c.width * 2, c.out_ch), dtype=torch.bfloat16, device="cuda")
        with pytest.raises(uf.UFError) as e:
            uf.uf_cmn_step(net, z, 2, out)                 # parameters never set
        assert e.value.code == uf.binding.UF_ERR_STATE
        with pytest.raises(uf.UFError) as e:
            uf.uf_cmn_set_param(net, "nope", np.zeros(4, np.uint16))
        assert e.value.code == uf.binding.UF_ERR_INVALID_ARG
        with pytest.raises(uf.UFError) as e:
            uf.uf_cmn_set_param(net, "s0.b0.skip", np.zeros((64, 64, 1, 1), np.uint16), np.zeros(64, np.float32))
        assert e.value.code == uf.binding.UF_ERR_INVALID_ARG
    finally:
        uf.uf_cmn_destroy(net)


def test_cmn_step_with_another_device_current():
    """every uf_cmn_* call makes the handle's device current itself, and the dynamic-shared-memory limit of
    the convolution kernel is raised per handle (it is a per-device attribute).  Needs two GPUs: a handle on cuda:1 is
    set up and stepped while cuda:0 is current and must give the bits of a handle on cuda:0."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    c = wl.CMN_CONFIGS["cmn_tiny"]
    zb = wl.cmn_frames(c, 0, 2)
    outs = []
    for dev in (0, 1):
        torch.cuda.set_device(0)
        net = hz.CmnCuda(c, frames_max=2, device=dev)
        try:
            torch.cuda.set_device(0)
            outs.append(net.step(zb))
            torch.cuda.set_device(0)
            net.memory(0, 0)                              # a getter with the other device current
        finally:
            net.close()
    assert np.array_equal(outs[0], outs[1])
