"""CPU oracle for the causal memory network (streaming latent upsampler / HR decoder) of Ultra Flash
(SURVEY.md section 8(f) NEXT-4): paper section 2.2, Eq. 2, Algorithm 2 variants A and B
(P:472-552), configurations P:345-347.

*** TEST INFRASTRUCTURE — NOT A PRODUCT PATH ***  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It shares no code with the CUDA path
(paper_2606_09150_b200/csrc/uf_cmn*.cu) and imports nothing from the package.

What the paper fixes
  * CausalMemBlock, Eq. 2:
        h_t^(l) = relu( Conv3(Conv2(relu(Conv1([h_t^(l-1) ; m_{t-1}^(l)])))) + W_skip h_t^(l-1) )
    all three convolutions 3x3, W_skip a 1x1 projection, [.;.] channel concatenation.
  * The network (Alg. 2 lines 4-18 / 25-40): input 3x3 convolution, then per stage s: N_b blocks,
    PixelShuffle_{r_s}(Conv3x3^{up_s}), if s_s > 1 a 1x1 convolution that lifts the channels by s_s followed by a
    channel-to-time reshape, a 1x1 channel transition Conv^{ch_s}; finally an output 3x3 convolution.
  * Variant A (parallel) takes the memory by a temporal shift, M_t = H_{t-1}, M_1 = 0; variant B
    (streaming) keeps one memory per block, initialised to zero.

Readings (R-41 ... R-46; the paper is silent or at odds with itself)
  R-41  WHAT the memory is.  Variant A line 7 shifts the block INPUT (M_t = H_{t-1} with H the tensor entering the
        block); variant B line 31 stores h AFTER line 30, i.e. the block OUTPUT.  The two differ, and only the
        first one can be evaluated "all frames simultaneously" and makes the "parallel (training) and
        sequential (streaming inference) execution modes" the same function.  Taken: m_t^(l) = h_t^(l-1),
        the block's input at the previous frame of the block's own frame rate; the first frame of a stream sees
        zeros.  `forward_parallel` (A) and `CausalMemStream.step` (B) implement it independently and are pinned
        to agree frame by frame.  The literal variant B (memory = block OUTPUT) is available as
        `CausalMemStream(..., memory="output")`; it is a different function from the second frame on.
  R-42  Zero padding (spatial size is preserved by every 3x3 convolution); cross-correlation as in every deep
        learning framework: out[y,x,o] = b[o] + sum_{i,dy,dx} w[o,i,dy,dx] * in[y+dy-1, x+dx-1, i].
  R-43  Every convolution has a bias except W_skip (Eq. 2 writes it as a plain projection); no activation other
        than the two ReLUs of Eq. 2.
  R-44  PixelShuffle_r (Shi et al. 2016, the usual convention): out[y*r+i, x*r+j, c] = in[y, x, c*r*r + i*r + j].
        Channel-to-time: frame f, channel k*C + c  ->  frame f*s + k, channel c (k = 0 .. s-1).
  R-45  Channels: stage s runs at stage_channels[s]; Conv^{ch_s} maps stage_channels[s] -> stage_channels[s+1]
        (the last one to stage_channels[-1] when the list has one more entry than stages, "[256,128,64,64]",
        else to itself, "[256,128,64]").  Note: with these widths one stage-1 block alone has 2.4 M weights,
        so P:345's "~2.1M parameters" and the latencies of Table 20 do not follow from P:345-347;
        the widths are taken, the totals are context.
  R-46  Arithmetic: bf16 storage between layers ("bf16 mixed precision"): inputs, weights and every layer
        output are bf16 values; inside a layer the sum is exact-ish (fp64 here, fp32 tensor-core accumulation on
        the GPU), bias (fp32 value) added, ReLU, then ONE rounding to bf16 (nearest even).  Conv3 and W_skip of a
        block are one sum, rounded once.  PixelShuffle and channel-to-time are permutations.

Tensors are float64 arrays holding bf16-representable values, layout [F, H, W, C] (frames, rows, columns,
channels); weights [C_out, C_in, 3, 3] or [C_out, C_in] (1x1).
"""
from __future__ import annotations

import dataclasses

import numpy as np


# ---- bf16 rounding (the one storage format, R-46) ------------------------------------------------------------
def round_bf16(x: np.ndarray) -> np.ndarray:
    """fp64 -> nearest bf16 (ties to even), returned as fp64.  ONE rounding, straight from the fp64 value (going
    through fp32 first would round twice)."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    flat = x.reshape(-1)
    m, e = np.frexp(flat)                       # flat = m * 2^e, 0.5 <= |m| < 1
    e_min = -125                                # smallest normal exponent in frexp convention (2^-126 = 0.5 * 2^-125)
    e_eff = np.maximum(e, e_min)                # subnormals: fixed quantum
    q = np.ldexp(1.0, e_eff - 8)                # spacing of the bf16 numbers (8 significant bits) in that binade
    with np.errstate(invalid="ignore"):
        r = np.rint(flat / q) * q               # rint = ties to even; flat / q and * q are exact (powers of two)
    bad = ~np.isfinite(flat)
    r[bad] = flat[bad]
    out = r.reshape(x.shape)
    big = np.abs(out) >= 2.0 ** 128
    out[big] = np.sign(out[big]) * np.inf
    return out


# ---- the primitive layers, written from their definitions (R-42, R-44) -----------------------------------------
def conv3x3(x: np.ndarray, w: np.ndarray, b: np.ndarray | None) -> np.ndarray:
    """x [F,H,W,Ci], w [Co,Ci,3,3], b [Co] -> [F,H,W,Co]; zero padding, cross-correlation (R-42).  fp64, unrounded."""
    F, H, W, Ci = x.shape
    Co = w.shape[0]
    assert w.shape == (Co, Ci, 3, 3)
    xp = np.zeros((F, H + 2, W + 2, Ci), dtype=np.float64)
    xp[:, 1:H + 1, 1:W + 1, :] = x
    out = np.zeros((F, H, W, Co), dtype=np.float64)
    for dy in range(3):
        for dx in range(3):
            out += xp[:, dy:dy + H, dx:dx + W, :] @ w[:, :, dy, dx].T
    if b is not None:
        out += b
    return out


def conv1x1(x: np.ndarray, w: np.ndarray, b: np.ndarray | None) -> np.ndarray:
    out = x @ w.T
    if b is not None:
        out = out + b
    return out


def pixel_shuffle(x: np.ndarray, r: int) -> np.ndarray:
    """[F,H,W,C*r*r] -> [F,H*r,W*r,C], out[y*r+i, x*r+j, c] = in[y, x, c*r*r + i*r + j] (R-44)"""
    F, H, W, Crr = x.shape
    C = Crr // (r * r)
    assert C * r * r == Crr
    return x.reshape(F, H, W, C, r, r).transpose(0, 1, 4, 2, 5, 3).reshape(F, H * r, W * r, C)


def channel_to_time(x: np.ndarray, s: int) -> np.ndarray:
    """[F,H,W,s*C] -> [F*s,H,W,C], frame f*s+k, channel c = in frame f, channel k*C + c (R-44)"""
    F, H, W, sC = x.shape
    C = sC // s
    assert C * s == sC
    return x.reshape(F, H, W, s, C).transpose(0, 3, 1, 2, 4).reshape(F * s, H, W, C)


def relu(x):
    return np.maximum(x, 0.0)


# ---- configuration and weights ----------------------------------------------------------------------------------
@dataclasses.dataclass(frozen=True)
class CmnConfig:
    in_ch: int
    out_ch: int
    stage_channels: tuple          # one per stage (+ optionally the width after the last channel transition)
    n_blocks: int                  # N_b CausalMemBlocks per stage
    spatial_factors: tuple         # r_s
    temporal_factors: tuple        # s_s

    @property
    def n_stages(self) -> int:
        return len(self.spatial_factors)

    def ch_out(self, s: int) -> int:
        """width after Conv^{ch_s} (R-45)"""
        if s + 1 < len(self.stage_channels):
            return self.stage_channels[s + 1]
        return self.stage_channels[s]


UPSAMPLER = CmnConfig(16, 16, (256, 128, 64), 3, (2, 1, 1), (1, 1, 1))
HR_DECODER = CmnConfig(16, 3, (256, 128, 64, 64), 3, (2, 2, 2), (1, 2, 2))


def weight_names(cfg: CmnConfig):
    """(name, shape) of every parameter in network order; biases are `<name>.b`"""
    out = [("in", (cfg.stage_channels[0], cfg.in_ch, 3, 3))]
    for s in range(cfg.n_stages):
        c = cfg.stage_channels[s]
        for b in range(cfg.n_blocks):
            p = f"s{s}.b{b}."
            out += [(p + "c1", (c, 2 * c, 3, 3)), (p + "c2", (c, c, 3, 3)), (p + "c3", (c, c, 3, 3)),
                    (p + "skip", (c, c))]
        r, t = cfg.spatial_factors[s], cfg.temporal_factors[s]
        out.append((f"s{s}.up", (c * r * r, c, 3, 3)))
        if t > 1:
            out.append((f"s{s}.texp", (c * t, c)))
        out.append((f"s{s}.ch", (cfg.ch_out(s), c)))
    out.append(("out", (cfg.out_ch, cfg.ch_out(cfg.n_stages - 1), 3, 3)))
    return out


def has_bias(name: str) -> bool:
    return not name.endswith("skip")           # R-43


# ---- one CausalMemBlock, Eq. 2 with R-41/R-43/R-46 ---------------------------------------------------------------
def mem_block(h: np.ndarray, m: np.ndarray, wt: dict, p: str) -> np.ndarray:
    """h, m [F,H,W,C]: the block's input at frames t and t-1.  Returns the block's output (bf16 values)."""
    a = round_bf16(relu(conv3x3(np.concatenate([h, m], axis=-1), wt[p + "c1"], wt[p + "c1.b"])))
    a = round_bf16(conv3x3(a, wt[p + "c2"], wt[p + "c2.b"]))
    a = conv3x3(a, wt[p + "c3"], wt[p + "c3.b"]) + conv1x1(h, wt[p + "skip"], None)
    return round_bf16(relu(a))


def _stage_tail(h: np.ndarray, cfg: CmnConfig, s: int, wt: dict) -> np.ndarray:
    """PixelShuffle(Conv^up), temporal expansion, channel transition (Alg. 2 lines 12-16 / 34-38)"""
    r, t = cfg.spatial_factors[s], cfg.temporal_factors[s]
    h = round_bf16(conv3x3(h, wt[f"s{s}.up"], wt[f"s{s}.up.b"]))
    if r > 1:
        h = pixel_shuffle(h, r)
    if t > 1:
        h = channel_to_time(round_bf16(conv1x1(h, wt[f"s{s}.texp"], wt[f"s{s}.texp.b"])), t)
    return round_bf16(conv1x1(h, wt[f"s{s}.ch"], wt[f"s{s}.ch.b"]))


# ---- Variant A: all frames at once, memory by temporal shift --------------------------------------
def forward_parallel(z: np.ndarray, cfg: CmnConfig, wt: dict) -> np.ndarray:
    """z [T,H,W,in_ch] (the whole stream) -> [T*prod(s), H*prod(r), W*prod(r), out_ch]"""
    h = round_bf16(conv3x3(z, wt["in"], wt["in.b"]))
    for s in range(cfg.n_stages):
        for b in range(cfg.n_blocks):
            m = np.zeros_like(h)
            m[1:] = h[:-1]                                   # M_t = H_{t-1}, M_1 = 0 (line 7)
            h = mem_block(h, m, wt, f"s{s}.b{b}.")
        h = _stage_tail(h, cfg, s, wt)
    return round_bf16(conv3x3(h, wt["out"], wt["out.b"]))


# ---- Variant B: streaming, explicit memory per block ----------------------------------------------
class CausalMemStream:
    """State = one memory frame per block (zeros at the start of a stream).  `step` takes the next frames of the
    stream (any number; a chunk) and emits their outputs; frame by frame inside (Alg. 2 line 24)."""

    def __init__(self, cfg: CmnConfig, wt: dict, memory: str = "input"):
        """memory = "input" (default, R-41: what the GPU path and `forward_parallel` compute): a block remembers its
        INPUT at the previous frame, Alg. 2 variant A line 7 carried into the streaming loop.
        memory = "output": Alg. 2 variant B exactly as printed: the memory is overwritten
        with h AFTER the block's ReLU, i.e. the block's OUTPUT.  That is a recurrence over frames (every earlier frame
        reaches the current one), cannot be evaluated for all frames at once, and is NOT the function variant A
        defines; it exists here so that the difference between the two readings is a number, not an argument."""
        if memory not in ("input", "output"):
            raise ValueError(memory)
        self.cfg, self.wt, self.memory = cfg, wt, memory
        self.mem: dict[str, np.ndarray | None] = {}
        self.reset()

    def reset(self):
        self.mem = {f"s{s}.b{b}.": None for s in range(self.cfg.n_stages) for b in range(self.cfg.n_blocks)}

    def _frames(self, h: np.ndarray, s: int, b0: int) -> np.ndarray:
        """run frames of h (at the current stage's frame rate) through blocks b0.. of stage s one frame at a time"""
        outs = []
        for f in range(h.shape[0]):
            x = h[f:f + 1]
            for b in range(b0, self.cfg.n_blocks):
                p = f"s{s}.b{b}."
                m = self.mem[p] if self.mem[p] is not None else np.zeros_like(x)
                if self.memory == "input":
                    self.mem[p] = x                          # R-41: the block's input is the next frame's memory
                x = mem_block(x, m, self.wt, p)
                if self.memory == "output":
                    self.mem[p] = x                          # variant B lines 31-32 as printed: m <- h after the ReLU
            outs.append(x)
        return np.concatenate(outs, axis=0)

    def step(self, z: np.ndarray) -> np.ndarray:
        outs = []
        for f in range(z.shape[0]):                          # "for each incoming frame" (line 24)
            h = round_bf16(conv3x3(z[f:f + 1], self.wt["in"], self.wt["in.b"]))
            for s in range(self.cfg.n_stages):
                h = self._frames(h, s, 0)                    # a frame expanded in time upstream arrives as several
                h = _stage_tail(h, self.cfg, s, self.wt)
            outs.append(round_bf16(conv3x3(h, self.wt["out"], self.wt["out.b"])))
        return np.concatenate(outs, axis=0)


def flop_count(cfg: CmnConfig, H: int, W: int, frames: int) -> int:
    """2 * multiply-adds of all convolutions for `frames` input frames of H x W (the definition's count: real
    channel numbers, no padding)"""
    total = 0
    px = H * W * frames
    shapes = dict(weight_names(cfg))
    total += px * int(np.prod(shapes["in"]))
    for s in range(cfg.n_stages):
        for b in range(cfg.n_blocks):
            for k in ("c1", "c2", "c3", "skip"):
                total += px * int(np.prod(shapes[f"s{s}.b{b}.{k}"]))
        total += px * int(np.prod(shapes[f"s{s}.up"]))
        px *= cfg.spatial_factors[s] ** 2
        if cfg.temporal_factors[s] > 1:
            total += px * int(np.prod(shapes[f"s{s}.texp"]))
            px *= cfg.temporal_factors[s]
        total += px * int(np.prod(shapes[f"s{s}.ch"]))
    total += px * int(np.prod(shapes["out"]))
    return 2 * total
