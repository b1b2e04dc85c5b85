"""GPU parity of the cache window policy (NEXT-3): the usage statistic the select kernel counts, the window the host
function derives from it, and the slot maps that follow, against oracle/uf_window_policy.py — bit-exact."""
import numpy as np
import pytest

import uf_workloads as wl
import uf_harness as hz
from oracle import uf_window_policy as wp

pytestmark = pytest.mark.gpu


def _weak_keys(Kb, factor):
    """scale a chunk's keys by an exactly representable factor (-1: the positional part then scores NEGATIVE against
    every query block, so no row ever picks one of its blocks)"""
    k = wl.bf16_bits_to_f32(Kb) * np.float32(factor)
    return wl.f32_to_bf16_bits(k)


def test_content_policy_stream_matches_oracle():
    """12 chunks, capacity 4, top 30 %: chunks 2 and 7 carry negated keys (never among the top-k), so when one of
    them becomes the oldest survivor its share of the kept blocks is 0 and it is evicted one append before FIFO
    would; otherwise the window grows back to C.  Usage counts, windows, slot maps, indices and outputs all match the oracle."""
    import paper_2606_09150_b200 as uf
    w = wl.scaled(wl.CONFIGS["1k"], "winpol", n_heads=2, frames_per_chunk=1, grid_h=24, grid_w=27, capacity_chunks=4,
                  topk_percent=30)
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    kw = dict(compact_window=2, min_share_permille=150)
    dropped_early = 0
    try:
        for c in range(12):
            W = uf.uf_next_window(cu.ctx, uf.UF_WIN_CONTENT, stream=cu.stream, **kw)
            Wo = wp.next_window(orc, wp.CONTENT, **kw)
            assert W == Wo, f"chunk {c}: window {W} != oracle {Wo}"
            Qb, Kb, Vb = wl.make_chunk(w, c)
            if c in (2, 7):
                Kb = _weak_keys(Kb, -1.0)
            got = cu.step(Qb, Kb, Vb, topk_percent=30, window=W)
            ref = hz.oracle_step(orc, Qb, Kb, Vb, topk_percent=30, window=W)
            hz.compare_step(got, ref, f"[winpol chunk {c}]")
            kept, ids = uf.uf_get_select_usage(cu.ctx, cu.stream)
            kept_o, ids_o = wp.select_usage(orc)
            assert (kept, ids) == (kept_o, ids_o), f"chunk {c}: usage {kept} {ids} != oracle {kept_o} {ids_o}"
            n_res = got["slot_map"][1]
            dropped_early += int(n_res < min(c + 1, w.capacity_chunks))
        assert dropped_early > 0, "the weak chunks must have been dropped before the FIFO would have"
    finally:
        cu.close()


def test_usage_statistic_in_paper_mode():
    import paper_2606_09150_b200 as uf
    w = wl.scaled(wl.CONFIGS["1k_paper"], "winpaper", n_heads=2, frames_per_chunk=3, grid_h=20, grid_w=27,
                  capacity_chunks=3, window=3)
    cu, orc = hz.PaperCudaStream(w), hz.make_paper_oracle(w)
    try:
        for c in range(4):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            got = cu.step(Qb, Kb, Vb, topk_count=6)
            ref = hz.paper_oracle_step(orc, Qb, Kb, Vb, topk_count=6)
            hz.compare_paper_step(got, ref, f"[winpaper chunk {c}]")
            assert uf.uf_get_select_usage(cu.ctx, cu.stream) == wp.select_usage(orc)
            assert uf.uf_next_window(cu.ctx, uf.UF_WIN_CONTENT, compact_window=1, min_share_permille=100, stream=cu.stream) \
                == wp.next_window(orc, wp.CONTENT, compact_window=1, min_share_permille=100)
    finally:
        cu.close()


def test_position_and_memory_policies_on_device_ctx():
    import paper_2606_09150_b200 as uf
    w = wl.scaled(wl.CONFIGS["1k"], "winpos", n_heads=1, frames_per_chunk=1, grid_h=16, grid_w=16, capacity_chunks=3)
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    try:
        for c in range(6):
            W = uf.uf_next_window(cu.ctx, uf.UF_WIN_POSITION, warm_chunks=3, compact_window=2)
            assert W == wp.next_window(orc, wp.POSITION, warm_chunks=3, compact_window=2) == (3 if c < 3 else 2)
            Qb, Kb, Vb = wl.make_chunk(w, c)
            got = cu.step(Qb, Kb, Vb, topk_count=1, window=W)
            ref = hz.oracle_step(orc, Qb, Kb, Vb, topk_count=1, window=W)
            hz.compare_step(got, ref, f"[winpos chunk {c}]")
        sb = wp.slot_bytes(orc)
        assert sb == 2 * 1 * 2 * 128 * 128 * 2
        assert uf.uf_next_window(cu.ctx, uf.UF_WIN_MEMORY, budget_bytes=2 * sb + 5) == 2
    finally:
        cu.close()
