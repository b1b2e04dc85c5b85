"""GPU parity of the CTA-pair attention kernel (uf_set_attn_impl(ctx, 2): cta_group::2 MMAs over two CTAs, one query
tile per CTA, triple-buffered S, two softmax warp groups per CTA taking the key blocks in turn with one shared reference
max per row) against the fp64 oracle, on the cases that exercise what is specific to it: an odd
number of query blocks (the second CTA of the last pair has no tile), blocks only one tile of a pair attends
(zero-fill steps), the deferred raise of the reference max with the tensor pipe up to two blocks behind, the
exact-max redo kernel, and BASELINE.json configs[1] at full size (every row against the default kernel, sampled
(head, query block) pairs against the oracle).  The whole of tests/test_gpu_parity.py also runs on this kernel with
UF_TEST_ATTN_IMPL=2 (tests/uf_harness.py)."""
import numpy as np
import pytest

import uf_workloads as wl
import uf_harness as hz
from test_gpu_parity import _oracle_attn_parallel, _run_stream

pytestmark = pytest.mark.gpu

PAIR = 2


def test_pair_small_stream_odd_blocks_ragged_tail():
    w = wl.scaled(wl.CONFIGS["1k"], "pair128", n_heads=2, frames_per_chunk=1, grid_h=23, grid_w=24,
                  capacity_chunks=3, topk_percent=50)
    assert w.bpc == 5                                        # last pair: one tile, 40-token tail
    _run_stream(w, wl.make_stream(w, 6), topk_percent=50, impl=PAIR)


def test_pair_few_candidates_mostly_single_tile_entries():
    # top-1 of few candidates: neighbouring query blocks rarely agree, so most merged entries belong to one tile
    w = wl.scaled(wl.CONFIGS["1k"], "pair128k1", n_heads=3, frames_per_chunk=1, grid_h=32, grid_w=32, capacity_chunks=4,
                  amp=0.0)
    _run_stream(w, wl.make_stream(w, 5), topk_count=1, impl=PAIR)


@pytest.mark.parametrize("scale", [0.3, 8.0])
def test_pair_sharp_softmax(scale):
    w = wl.scaled(wl.CONFIGS["1k"], "pairsharp", n_heads=2, frames_per_chunk=1, grid_h=20, grid_w=29,
                  capacity_chunks=3, topk_percent=50)
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    try:
        redone = 0
        for c in range(3):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            got = cu.step(Qb, Kb, Vb, topk_percent=50, scale=scale, impl=PAIR)
            redone += cu.uf.uf_attn_redone_items(cu.ctx, cu.stream)
            ref = hz.oracle_step(orc, Qb, Kb, Vb, topk_percent=50, scale=scale)
            hz.compare_step(got, ref, f"[pair sharp scale {scale} chunk {c}]")
        if scale >= 8.0:
            assert redone > 0, "scale 8 must overflow the stale-max exponentials and take the exact-max kernel"
    finally:
        cu.close()


def test_pair_full_size_1k():
    import torch
    w = wl.CONFIGS["1k"]
    nqb = w.bpc
    rng = np.random.default_rng(7)
    sampled = sorted({0, 1, nqb - 2, nqb - 1} | set(int(x) for x in rng.integers(0, nqb, 8)))
    jobs = [(int(h), sampled) for h in (0, 5, w.n_heads - 1)]
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    try:
        for c in range(w.prior_chunks + 1):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            got = cu.step(Qb, Kb, Vb, topk_percent=w.topk_percent, impl=PAIR)
            ref = hz.oracle_step(orc, Qb, Kb, Vb, topk_percent=w.topk_percent, attn=False)
            hz.compare_step(got, ref, f"[pair 1k chunk {c}]")
        assert not np.isnan(got["O"]).any() and np.isfinite(got["lse"]).all()
        assert cu.uf.uf_attn_redone_items(cu.ctx, cu.stream) == 0
        # every row against the default tcgen05 kernel on the same selection
        q = cu.to_dev(Qb)
        o0 = torch.empty_like(q)
        n, H, d = Qb.shape
        cu.uf.uf_set_attn_impl(cu.ctx, 0)
        cu.uf.uf_sparse_attn_fwd(cu.ctx, q, o0, None, n, H * d, d, 0.0, cu.stream)
        torch.cuda.synchronize()
        diff = (o0.float() - torch.from_numpy(got["O"]).to(o0.device)).abs()
        assert float(diff.max()) <= hz.O_MAX_ABS and float(diff.mean()) <= hz.O_MEAN_ABS, (float(diff.max()), float(diff.mean()))
        ref["O"], ref["lse"] = _oracle_attn_parallel(orc, hz.bits_to_f64(Qb), jobs)
        hz.compare_step(got, ref, "[pair 1k attention]")
    finally:
        cu.close()
