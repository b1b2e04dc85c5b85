"""Seeded synthetic workloads for the Ultra Flash sparse causal chunk attention path.

This module holds ONLY input generation (shapes, seeds, value distributions, bf16
rounding).  It contains none of the method's arithmetic (no pooling, scoring, top-k,
softmax or cache policy) and imports neither `oracle/` nor the CUDA package: it is the
one module both sides may share (tests and bench.py feed its arrays to both).

Shapes follow BASELINE.json `configs[0..4]`; the value recipe is SURVEY.md §8(d)
(stated again in DESIGN.md §"Input recipe"): Q/K = N(0,1) + A * smooth sinusoidal
(t,h,w) positional features, V = N(0,1), rounded to bf16 (round-to-nearest-even).
The paper's real workloads are DiT activations of a trained Wan2.1-1.3B-shaped SR model
 which do not exist here; these inputs stand in for them.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np


@dataclasses.dataclass(frozen=True)
class Workload:
    """One BASELINE.json config.  `prior_chunks` = chunks appended before the timed one."""
    name: str
    n_heads: int
    head_dim: int
    block: int
    frames_per_chunk: int          # latent frames per chunk (F)
    grid_h: int                    # token grid height (Hg) after VAE /8 and 2x2 patchify
    grid_w: int                    # token grid width  (Wg)
    capacity_chunks: int           # C: resident non-sink chunks incl. the current one
    prior_chunks: int              # chunks in the stream before the measured chunk
    topk_count: int                # >=0: exact count; -1: use percent
    topk_percent: int              # percent of |CAND|
    amp: float                     # positional amplitude A
    sink_blocks: int = 1
    k_min: int = 4                 # PAPER.md:818 (k_min = 4), floor in percent mode only
    n_stream_chunks: int = 0       # >0: rolling-stream config (config 3)
    # paper-mask variants: 3-D tiles of the chunk's token grid, r x r block window, rho
    tile: tuple | None = None      # (b_t, b_h, b_w), PAPER.md:343 (2, 8, 8); None = flat blocks (BASELINE.json)
    window: int = 9                # PAPER.md:343 "local window 9 x 9"
    rho_permille: int = 1000       # PAPER.md:343 rho = 1.0

    @property
    def tile_grid(self) -> tuple[int, int, int]:
        """(nbt, nbh, nbw): tiles per chunk along t, y, x (edge tiles ragged)"""
        bt, bh, bw = self.tile
        return -(-self.frames_per_chunk // bt), -(-self.grid_h // bh), -(-self.grid_w // bw)

    @property
    def n_tiles(self) -> int:
        a, b, c = self.tile_grid
        return a * b * c

    @property
    def chunk_tokens(self) -> int:
        return self.frames_per_chunk * self.grid_h * self.grid_w

    @property
    def bpc(self) -> int:
        return -(-self.chunk_tokens // self.block)


def token_grid(height_px: int, width_px: int, vae: int = 8, patch: int = 2) -> tuple[int, int]:
    """Token grid (Hg, Wg) of one latent frame: pixels / VAE stride / spatial patch.
    PAPER.md:343 ("patch size (1,2,2)"), 8x spatial VAE (BASELINE.json configs[1])."""
    return height_px // vae // patch, width_px // vae // patch


_G1K = token_grid(1088, 1920)   # (68, 120) -> 8160 tokens / latent frame
_G2K = token_grid(1440, 2560)   # (90, 160) -> 14400 tokens / latent frame

CONFIGS: dict[str, Workload] = {
    # configs[0]: tiny, 1 head x 64, 3 chunks of 2 frames x 8x8 tokens, block 64, top-2, cache holds all
    "tiny": Workload("tiny", 1, 64, 64, 2, 8, 8, capacity_chunks=3, prior_chunks=2,
                     topk_count=2, topk_percent=-1, amp=0.0, n_stream_chunks=3),
    # configs[1]: 1K step, 1 prior chunk + sink => C = 2
    "1k": Workload("1k", 12, 128, 128, 3, _G1K[0], _G1K[1], capacity_chunks=2, prior_chunks=1,
                   topk_count=-1, topk_percent=25, amp=2.0),
    # configs[2]: 2K step, 2 prior chunks + sink => C = 3
    "2k": Workload("2k", 12, 128, 128, 3, _G2K[0], _G2K[1], capacity_chunks=3, prior_chunks=2,
                   topk_count=-1, topk_percent=15, amp=2.0),
    # configs[3]: 1K rolling stream, 20 chunks, capacity 3 + sink, top 25 %
    "1k_stream": Workload("1k_stream", 12, 128, 128, 3, _G1K[0], _G1K[1], capacity_chunks=3,
                          prior_chunks=2, topk_count=-1, topk_percent=25, amp=2.0,
                          n_stream_chunks=20),
    # configs[4]: wide model, 40 heads, 2 prior chunks + sink, top 20 %, amplitude 3
    "wide": Workload("wide", 40, 128, 128, 3, _G1K[0], _G1K[1], capacity_chunks=3, prior_chunks=2,
                     topk_count=-1, topk_percent=20, amp=3.0),
    # paper-mask variants of configs[1] / configs[2]: same grids, heads, chunking and cache as BASELINE.json, but the
    # mask of PAPER.md section 2.3.1 (tiles (2,8,8), 9 x 9 window as an intersection, budget from the repaired Eq. 10
    # at rho = 1.0, no sink).  1K: 2 x 9 x 15 = 270 tiles per chunk, 2K: 2 x 12 x 20 = 480.
    "1k_paper": Workload("1k_paper", 12, 128, 128, 3, _G1K[0], _G1K[1], capacity_chunks=2, prior_chunks=1,
                         topk_count=-1, topk_percent=-1, amp=2.0, sink_blocks=0, tile=(2, 8, 8)),
    "2k_paper": Workload("2k_paper", 12, 128, 128, 3, _G2K[0], _G2K[1], capacity_chunks=3, prior_chunks=2,
                         topk_count=-1, topk_percent=-1, amp=2.0, sink_blocks=0, tile=(2, 8, 8)),
    # the paper's OWN chunking: "streaming chunk size: 2 latent frames" at 960 x 1664
    # -> 60 x 104 tokens per latent frame, 12 480 tokens per chunk, "KV cache: 3 temporal windows".  The
    # (2,8,8) tiles are then full in t and 94 % full overall (1 x 8 x 13 = 104 tiles per chunk; only the last tile row
    # is ragged: 60 = 7 * 8 + 4), the configuration section 2.3.1 was written for; BASELINE.json's 3-frame chunks leave
    # half of the temporal tiles with one frame of two.
    "1k_paper_native": Workload("1k_paper_native", 12, 128, 128, 2, *token_grid(960, 1664), capacity_chunks=3,
                                prior_chunks=2, topk_count=-1, topk_percent=-1, amp=2.0, sink_blocks=0, tile=(2, 8, 8)),
}


def scaled(w: Workload, name: str, **kw) -> Workload:
    """A smaller/other variant of a workload with the same recipe (for CPU-seconds parity cases)."""
    return dataclasses.replace(w, name=name, **kw)


# ---------------------------------------------------------------------------
# bf16 <-> fp32 format conversion (a storage format, not method arithmetic)
# ---------------------------------------------------------------------------

def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round float32 to bf16 (round-to-nearest-even); returns uint16 bit patterns."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    rnd = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + rnd) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """Exact widening of bf16 bit patterns to float32."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


# ---------------------------------------------------------------------------
# Positional features and chunk generator
# ---------------------------------------------------------------------------

def _pos_tables(w: Workload):
    """Frequencies / phases drawn once per run from default_rng(10_000) in the order
    f_t, f_h, f_w, phi."""
    g = np.random.default_rng(10_000)
    d, H = w.head_dim, w.n_heads
    f_t = g.integers(0, 2, d)
    f_h = g.integers(0, 3, d)
    f_w = g.integers(0, 3, d)
    phi = g.uniform(0.0, 2.0 * math.pi, (H, d))
    return f_t, f_h, f_w, phi


def positional(w: Workload, chunk: int, n_tokens: int | None = None) -> np.ndarray:
    """p[n, h, j] = sin(2*pi*(f_t[j]*t/24 + f_h[j]*y/Hg + f_w[j]*x/Wg) + phi[h, j]), float32,
    tokens in raster (t, y, x) order with t = chunk*F + n // (Hg*Wg).
    Evaluated as sin(a)cos(phi) + cos(a)sin(phi) in float64, then cast to float32."""
    N = w.chunk_tokens if n_tokens is None else n_tokens
    f_t, f_h, f_w, phi = _pos_tables(w)
    n = np.arange(N)
    per_frame = w.grid_h * w.grid_w
    t = chunk * w.frames_per_chunk + n // per_frame
    y = (n % per_frame) // w.grid_w
    x = n % w.grid_w
    a = 2.0 * math.pi * (np.outer(t / 24.0, f_t) + np.outer(y / w.grid_h, f_h) + np.outer(x / w.grid_w, f_w))
    sa, ca = np.sin(a), np.cos(a)                               # [N, d]
    p = sa[:, None, :] * np.cos(phi)[None] + ca[:, None, :] * np.sin(phi)[None]
    return p.astype(np.float32)


def make_chunk(w: Workload, chunk: int, seed: int | None = None, n_tokens: int | None = None,
               rng: np.random.Generator | None = None):
    """Q, K, V of one chunk as bf16 bit patterns, uint16 [N, H, d].

    Seed rule: chunk c of a stream uses seed c unless `rng` is given (config 0
    draws all chunks in order from one default_rng(0)).  Draw order: Qn, Kn, Vn."""
    N = w.chunk_tokens if n_tokens is None else n_tokens
    if rng is None:
        rng = np.random.default_rng(chunk if seed is None else seed)
    shape = (N, w.n_heads, w.head_dim)
    qn = rng.standard_normal(shape, dtype=np.float32)
    kn = rng.standard_normal(shape, dtype=np.float32)
    vn = rng.standard_normal(shape, dtype=np.float32)
    if w.amp != 0.0:
        p = positional(w, chunk, N)
        qn += np.float32(w.amp) * p
        kn += np.float32(w.amp) * p
    return f32_to_bf16_bits(qn), f32_to_bf16_bits(kn), f32_to_bf16_bits(vn)


def make_stream(w: Workload, n_chunks: int):
    """List of (Q, K, V) bf16-bit chunks 0..n_chunks-1.  'tiny' draws from one rng(0) in order."""
    if w.name.startswith("tiny"):
        rng = np.random.default_rng(0)
        return [make_chunk(w, c, rng=rng) for c in range(n_chunks)]
    return [make_chunk(w, c) for c in range(n_chunks)]


# ---------------------------------------------------------------------------
# Model state for the fused QK-norm + RoPE + append step: inputs, like weights
# ---------------------------------------------------------------------------

ROPE_AXIS_DIMS = (44, 42, 42)        # PAPER.md:343 "3D RoPE with axis dims (44,42,42)"


def rope_tables(max_pos: int, dims=ROPE_AXIS_DIMS, theta: float = 10000.0):
    """cos / sin tables a Wan2.1-style model precomputes once: float32 [max_pos, d/2] (computed in fp64, stored in
    fp32); column i of the axis segment of dim D holds cos / sin(pos * theta**(-2 i / D)).  An INPUT of the step
    (both sides read the same numbers); the oracle states the definition they must satisfy
    (oracle/uf_rope_norm.py: rope_table) and a CPU test compares."""
    freq = np.concatenate([theta ** (-(2.0 * np.arange(D // 2, dtype=np.float64)) / D) for D in dims])
    ang = np.outer(np.arange(max_pos, dtype=np.float64), freq)
    return np.cos(ang).astype(np.float32), np.sin(ang).astype(np.float32)


def norm_weights(w: Workload, seed: int = 20_000):
    """RMSNorm weights of q and k, fp32 [H*d]: 1 + 0.1 N(0,1) (random-init stand-in for trained weights)"""
    g = np.random.default_rng(seed)
    n = w.n_heads * w.head_dim
    return ((1.0 + 0.1 * g.standard_normal(n)).astype(np.float32),
            (1.0 + 0.1 * g.standard_normal(n)).astype(np.float32))


# ---------------------------------------------------------------------------
# Causal memory network: shapes, random-init weights, input frames
# ---------------------------------------------------------------------------

@dataclasses.dataclass(frozen=True)
class CmnWorkload:
    """One causal-memory-network configuration on a latent grid.  Input generation only."""
    name: str
    in_ch: int
    out_ch: int
    stage_channels: tuple          # per stage (+ optionally the width after the last channel transition)
    n_blocks: int
    spatial_factors: tuple
    temporal_factors: tuple
    height: int                    # input latent grid
    width: int
    frames_per_chunk: int


# the streaming latent upsampler; input = the LR latent of BASELINE.json's 1K workload (the HR latent
# grid 136 x 240 of 1088 x 1920 halved), chunk = 3 latent frames as in BASELINE.json configs[1]
CMN_CONFIGS = {
    "cmn_tiny": CmnWorkload("cmn_tiny", 16, 16, (64, 64), 2, (2, 1), (1, 2), 12, 20, 2),
    "cmn_upsampler_1k": CmnWorkload("cmn_upsampler_1k", 16, 16, (256, 128, 64), 3, (2, 1, 1), (1, 1, 1), 68, 120, 3),
    # the HR decoder, on a quarter-area crop of the 1K HR latent (the full 136 x 240 input makes
    # 1088 x 1920 x 12 frames of 64-channel activations per chunk)
    "cmn_decoder_crop": CmnWorkload("cmn_decoder_crop", 16, 3, (256, 128, 64, 64), 3, (2, 2, 2), (1, 2, 2), 68, 120, 1),
    # PAPER.md:347 at full size: the whole 136 x 240 HR latent of the 1K workload, a chunk of 3 latent frames in ->
    # 12 frames of 1088 x 1920 x 3 out ("8x8x4 spatiotemporal decoding"; Table 20 "HR Decoder")
    "cmn_decoder_1k": CmnWorkload("cmn_decoder_1k", 16, 3, (256, 128, 64, 64), 3, (2, 2, 2), (1, 2, 2), 136, 240, 3),
}


def cmn_param_shapes(c: CmnWorkload):
    """[(name, shape)] in network order; `<name>.b` biases exist for every entry except `*.skip`"""
    n_stages = len(c.spatial_factors)
    ch = list(c.stage_channels)
    out = [("in", (ch[0], c.in_ch, 3, 3))]
    for s in range(n_stages):
        for b in range(c.n_blocks):
            p = f"s{s}.b{b}."
            out += [(p + "c1", (ch[s], 2 * ch[s], 3, 3)), (p + "c2", (ch[s], ch[s], 3, 3)),
                    (p + "c3", (ch[s], ch[s], 3, 3)), (p + "skip", (ch[s], ch[s]))]
        r, t = c.spatial_factors[s], c.temporal_factors[s]
        out.append((f"s{s}.up", (ch[s] * r * r, ch[s], 3, 3)))
        if t > 1:
            out.append((f"s{s}.texp", (ch[s] * t, ch[s])))
        nxt = ch[s + 1] if s + 1 < len(ch) else ch[s]
        out.append((f"s{s}.ch", (nxt, ch[s])))
    last = ch[n_stages] if n_stages < len(ch) else ch[n_stages - 1]
    out.append(("out", (c.out_ch, last, 3, 3)))
    return out


def cmn_weights(c: CmnWorkload, seed: int = 30_000) -> dict:
    """Random-init stand-in for the trained network: every weight ~ N(0, gain / fan_in) rounded to bf16 (stored as
    float32 holding bf16 values), biases ~ 0.05 N(0,1) as float32.  gain 2 keeps ReLU activations O(1) through the
    depth (He init); W_skip and the 1x1 / output layers use gain 1."""
    g = np.random.default_rng(seed)
    wt = {}
    for name, shape in cmn_param_shapes(c):
        fan_in = int(np.prod(shape[1:]))
        gain = 2.0 if name.endswith(("c1", "c2", "in")) else 1.0
        w = g.standard_normal(shape).astype(np.float32) * np.float32(math.sqrt(gain / fan_in))
        wt[name] = bf16_bits_to_f32(f32_to_bf16_bits(w))
        if not name.endswith("skip"):
            wt[name + ".b"] = (0.05 * g.standard_normal(shape[0])).astype(np.float32)
    return wt


def cmn_frames(c: CmnWorkload, chunk: int, frames: int | None = None) -> np.ndarray:
    """bf16 bit patterns [F, H, W, in_ch] of chunk `chunk`: N(0,1) + a smooth field drifting over time (a latent video
    stand-in: neighbouring frames correlate, so the memory path matters)"""
    F = c.frames_per_chunk if frames is None else frames
    g = np.random.default_rng(40_000 + chunk)
    x = g.standard_normal((F, c.height, c.width, c.in_ch)).astype(np.float32) * np.float32(0.5)
    t = (chunk * c.frames_per_chunk + np.arange(F, dtype=np.float32))[:, None, None, None]
    yy = np.arange(c.height, dtype=np.float32)[None, :, None, None] / c.height
    xx = np.arange(c.width, dtype=np.float32)[None, None, :, None] / c.width
    ph = np.arange(c.in_ch, dtype=np.float32)[None, None, None, :]
    x += np.sin(2 * np.pi * (yy * (1 + ph % 3) + xx * (1 + ph % 2) + 0.05 * t) + ph).astype(np.float32)
    return f32_to_bf16_bits(x)


def scaled_cmn(c: CmnWorkload, name: str | None = None, **kw) -> CmnWorkload:
    """the same network on another grid / chunk length (CPU-seconds parity cases)"""
    return dataclasses.replace(c, name=name or c.name, **kw)
