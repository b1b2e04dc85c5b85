"""bench.py's FLOP accounting (the numerator of `value` and of `roofline.achieved`) against a direct enumeration of the
kept sets: 4 * d * sum over (head, query block) of valid query rows x valid kept keys.  CPU only:
the index lists come from the oracle here; on the GPU box bench.py feeds the same function with the library's lists."""
from __future__ import annotations

import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench  # noqa: E402
import uf_harness as hz  # noqa: E402
import uf_workloads as wl  # noqa: E402


def _enumerate_flop(orc, w, n_tok):
    total = 0
    for h in range(w.n_heads):
        for i in range(-(-n_tok // w.block)):
            rows = min((i + 1) * w.block, n_tok) - i * w.block
            keys = sum(orc.block_kv(g, fs)[0].shape[0] for g, fs in orc.kept_blocks(h, i))
            total += 4 * w.head_dim * rows * keys
    return total


def test_kept_flop_matches_enumeration_ragged_stream():
    w = wl.scaled(wl.CONFIGS["1k"], "acct", n_heads=2, head_dim=32, block=32, frames_per_chunk=1, grid_h=9, grid_w=11,
                  capacity_chunks=3, sink_blocks=1, topk_percent=40)
    orc = hz.make_oracle(w)
    n = w.chunk_tokens                                  # 99 tokens: 4 blocks, ragged tail of 3
    assert n == 99 and w.bpc == 4
    for c in range(4):
        Qb, Kb, Vb = wl.make_chunk(w, c)
        Q, K, V = hz.bits_to_f64(Qb), hz.bits_to_f64(Kb), hz.bits_to_f64(Vb)
        orc.kv_append(K, V)
        idx, cnt = orc.select_blocks(Q, -1, w.topk_percent)
        slot_map, _, newest = orc.slot_map()
        prior = {ch: n for ch in slot_map if ch >= 0}
        sink_tok = min(w.sink_blocks * w.block, n) if newest > 0 else 0
        got = bench.kept_flop(w, n, np.asarray(idx), sink_tok, prior)
        assert got == _enumerate_flop(orc, w, n), f"chunk {c}"


def test_kept_flop_full_size_closed_form():
    """configs[1] steady state: every query block keeps 48 full cache blocks + the 128-token sink + the whole chunk."""
    w = wl.CONFIGS["1k"]
    n, B, d, H = w.chunk_tokens, w.block, w.head_dim, w.n_heads
    nqb = -(-n // B)
    idx = np.tile(np.arange(48, dtype=np.int64)[None, None, :] + 1 * w.bpc, (H, nqb, 1))    # blocks 0..47 of chunk 1 (all full)
    got = bench.kept_flop(w, n, idx, B, {1: n, 2: n})
    assert got == 4 * d * H * n * (48 * B + B + n)
