"""GPU parity tests of paper-mask mode (3-D (2,8,8) tiles, 9 x 9 window as an intersection,
repaired Eq. 10) against oracle/uf_paper_mask.py, through the C ABI: kept block ids and counts bit-exact, outputs
within BASELINE.json's 2e-2 / 2e-3.  Run with `-m gpu` on a B200."""
from __future__ import annotations

import numpy as np
import pytest

import uf_workloads as wl
import uf_harness as hz

pytestmark = pytest.mark.gpu


def _small(name, **kw):
    base = dict(n_heads=2, frames_per_chunk=3, grid_h=20, grid_w=27, capacity_chunks=2, window=3)
    base.update(kw)
    return wl.scaled(wl.CONFIGS["1k_paper"], name, **base)


def _run(w, n_chunks, impl=0, windows=None, **sel):
    cu, orc = hz.PaperCudaStream(w), hz.make_paper_oracle(w)
    worst = (0.0, 0.0)
    try:
        for c in range(n_chunks):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            win = 0 if windows is None else windows[c]
            got = cu.step(Qb, Kb, Vb, window=win, impl=impl, **sel)
            ref = hz.paper_oracle_step(orc, Qb, Kb, Vb, window=win, **sel)
            r = hz.compare_paper_step(got, ref, f"[{w.name} chunk {c}]")
            worst = (max(worst[0], r[0]), max(worst[1], r[1]))
            assert (got["cnt"] >= 1).all() and (got["cnt"] <= got["k_eff"] + 1).all()
    finally:
        cu.close()
    return worst


def test_tile_untile_match_the_layout_contract():
    """uf_tile_tokens / uf_untile_tokens against the layout of include/uf.h written out in NumPy: valid rows carry
    their raster token, pad rows are zero, untile(tile(x)) == x and leaves nothing unwritten."""
    import torch
    w = _small("tile")
    cu = hz.PaperCudaStream(w)
    try:
        Qb, _, _ = wl.make_chunk(w, 0)
        t = cu.tile(Qb)
        torch.cuda.synchronize()
        tb = t.view(torch.int16).cpu().numpy().view(np.uint16)
        valid = cu.rows >= 0
        assert valid.sum() == w.chunk_tokens
        assert np.array_equal(tb[valid], Qb[cu.rows[valid]])
        assert not tb[~valid].any()
        n, H, d = Qb.shape
        back = torch.full((n, H, d), float("nan"), dtype=torch.bfloat16, device=cu.dev)
        cu.uf.uf_untile_tokens(cu.ctx, t, back, H * d, d, H * d, d, cu.stream)
        torch.cuda.synchronize()
        assert np.array_equal(back.view(torch.int16).cpu().numpy().view(np.uint16), Qb)
    finally:
        cu.close()


@pytest.mark.parametrize("impl", [0, 1])
def test_small_ragged_grid_count_mode(impl):
    """3 x 20 x 27 tokens -> 2 x 3 x 4 tiles, ragged along every axis (tiles of 128, 96, 64, 48, 24, ... tokens),
    window 3, exact count 5, capacity 2; tcgen05 kernel (impl 0) and CUDA-core kernel (impl 1)."""
    w = _small("p_small")
    assert w.n_tiles == 24
    _run(w, 4, impl=impl, topk_count=5)


def test_budget_mode_rho_and_window9():
    """tau_k from the repaired Eq. 10 at rho = 1.0 and 0.5 with the paper's 9 x 9 window on a 2 x 5 x 7 tile grid,
    capacity 3, odd number of tiles per chunk (the last query-tile pair has one tile)."""
    w = _small("p_rho", n_heads=3, grid_h=40, grid_w=51, capacity_chunks=3, window=9)
    assert w.n_tiles == 70
    _run(w, 4, rho_permille=1000)
    w2 = wl.scaled(w, "p_rho_half", grid_w=49)                       # 2 x 5 x 7, last column 1 token wide
    _run(w2, 3, rho_permille=500)


def test_dense_limit_and_zero_budget():
    """Window covering the grid and k >= N_blocks: every block of every resident chunk is kept (dense chunk-causal
    attention); k = 0: only the own block."""
    w = _small("p_dense", n_heads=1, window=99)
    _run(w, 3, topk_count=10_000)
    _run(w, 2, topk_count=0)


def test_window_shrink_in_paper_mode():
    w = _small("p_win", capacity_chunks=4)
    _run(w, 6, topk_count=6, windows=[0, 0, 0, 2, 4, 1])


def test_paper_mode_error_codes():
    import torch
    import paper_2606_09150_b200 as uf
    w = _small("p_err", n_heads=1)
    cu = hz.PaperCudaStream(w)
    try:
        Qb, Kb, Vb = wl.make_chunk(w, 0)
        q, k, v = cu.tile(Qb), cu.tile(Kb), cu.tile(Vb)
        with pytest.raises(uf.UFError) as ei:                          # raster-length chunk on a tiled ctx
            uf.uf_kv_append(cu.ctx, k, v, w.chunk_tokens, 128, 128, 0, cu.stream)
        assert ei.value.code == uf.binding.UF_ERR_INVALID_ARG
        uf.uf_kv_append(cu.ctx, k, v, cu.nt, 128, 128, 0, cu.stream)
        with pytest.raises(uf.UFError) as ei:                          # flat selection on a tiled ctx
            uf.uf_select_blocks(cu.ctx, q, cu.nt, 128, 128, 1, -1, None, None, cu.stream)
        assert ei.value.code == uf.binding.UF_ERR_STATE
        with pytest.raises(uf.UFError) as ei:                          # tiling a non-empty ctx
            uf.uf_ctx_set_tiling(cu.ctx, 3, 20, 27, 2, 8, 8, 9)
        assert ei.value.code == uf.binding.UF_ERR_STATE
        idx = torch.zeros((1, w.n_tiles, 2), dtype=torch.int32, device=cu.dev)
        with pytest.raises(uf.UFError) as ei:                          # idx rows too short for k' + 1
            uf.uf_select_blocks_paper(cu.ctx, q, cu.nt, 128, 128, 5, 1000, idx, 2, None, cu.stream)
        assert ei.value.code == uf.binding.UF_ERR_CAPACITY
    finally:
        cu.close()
    ctx = uf.uf_ctx_create(1, 128, 128, 24 * 128, 2, 1, 4, 0)          # a ctx with a sink cannot be tiled
    try:
        with pytest.raises(uf.UFError) as ei:
            uf.uf_ctx_set_tiling(ctx, 3, 20, 27, 2, 8, 8, 9)
        assert ei.value.code == uf.binding.UF_ERR_INVALID_ARG
    finally:
        uf.uf_ctx_destroy(ctx)
    ctx = uf.uf_ctx_create(1, 128, 128, 24 * 128, 2, 0, 4, 0)
    try:
        with pytest.raises(uf.UFError):                                # 2*8*4 != block
            uf.uf_ctx_set_tiling(ctx, 3, 20, 27, 2, 8, 4, 9)
        with pytest.raises(uf.UFError):                                # N_b * block != chunk_tokens_max
            uf.uf_ctx_set_tiling(ctx, 3, 20, 33, 2, 8, 8, 9)
        with pytest.raises(uf.UFError):                                # even window
            uf.uf_ctx_set_tiling(ctx, 3, 20, 27, 2, 8, 8, 8)
    finally:
        uf.uf_ctx_destroy(ctx)


@pytest.mark.parametrize("name", ["1k_paper", "2k_paper", "1k_paper_native"])
def test_full_size_paper_step(name):
    """BASELINE.json configs[1] / configs[2] under the paper's mask at full size, and the paper's own chunking
    (1k_paper_native: 2 latent frames of 60 x 104 tokens, 3 cached chunks, P:148 / P:343): ALL kept block ids and counts
    bit-exact; attention against the oracle on every row of two whole heads plus sampled tiles of two more; every
    row of every head against the CUDA-core kernel."""
    import torch
    w = wl.CONFIGS[name]
    NB = w.n_tiles
    rng = np.random.default_rng(2)
    jobs = [(h, list(range(lo, min(lo + 30, NB)))) for h in (0, w.n_heads - 1) for lo in range(0, NB, 30)]
    sampled = sorted({0, 1, NB - 2, NB - 1} | set(int(x) for x in rng.integers(0, NB, 8)))
    jobs += [(int(h), sampled) for h in rng.choice(np.arange(1, w.n_heads - 1), 2, replace=False)]
    cu, orc = hz.PaperCudaStream(w), hz.make_paper_oracle(w)
    try:
        for c in range(w.prior_chunks + 1):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            got = cu.step(Qb, Kb, Vb, rho_permille=w.rho_permille)
            ref = hz.paper_oracle_step(orc, Qb, Kb, Vb, rho_permille=w.rho_permille, attn=False)
            hz.compare_paper_step(got, ref, f"[{name} chunk {c}]")
        assert not np.isnan(got["O"]).any() and np.isfinite(got["lse"]).all()
        o2 = torch.empty_like(got["O_tiled"])
        H, d = w.n_heads, w.head_dim
        cu.uf.uf_set_attn_impl(cu.ctx, 1)
        cu.uf.uf_sparse_attn_fwd(cu.ctx, got["q_tiled"], o2, None, cu.nt, H * d, d, 0.0, cu.stream)
        torch.cuda.synchronize()
        valid = torch.from_numpy(cu.rows >= 0).to(o2.device)
        diff = (o2.float() - got["O_tiled"].float()).abs()[valid]
        assert float(diff.max()) <= hz.O_MAX_ABS and float(diff.mean()) <= hz.O_MEAN_ABS, (float(diff.max()), float(diff.mean()))
        O = np.full((w.chunk_tokens, H, d), np.nan)
        lse = np.full((H, w.chunk_tokens), np.nan)
        from concurrent.futures import ThreadPoolExecutor
        from threadpoolctl import threadpool_limits
        Q = hz.bits_to_f64(Qb)

        def run(job):
            h, tiles = job
            o, l = orc.sparse_attn(Q, heads=[h], qblocks=tiles)
            rows = np.concatenate([orc.tokens_of[i] for i in tiles])
            return h, rows, o[rows, h, :].copy(), l[h, rows].copy()

        with threadpool_limits(limits=2), ThreadPoolExecutor(8) as ex:
            for h, rows, o, l in ex.map(run, jobs):
                O[rows, h, :] = o
                lse[h, rows] = l
        ref["O"], ref["lse"] = O, lse
        r = hz.compare_paper_step(got, ref, f"[{name} attention]")
        kept = got["cnt"].astype(np.float64).mean()
        print(f"{name}: N_blocks {got['n_cand']}, tau_k {got['k_eff']}, mean kept blocks per row {kept:.1f}; "
              f"O max-abs {r[0]:.3e} mean-abs {r[1]:.3e}")
    finally:
        cu.close()
