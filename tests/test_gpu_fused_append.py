"""GPU parity of the fused QK-norm + 3-D RoPE + append + pooling step (NEXT-2, uf_qkv_rope_append) against the fp64
oracle oracle/uf_rope_norm.py: post-RoPE Q and cached K within ONE bf16 ulp of the fp64 definition (>= 99 % bit-equal),
cached V the input bits; then, teacher-forced on the kernel's own bf16 bits, the ordinary oracle: slot maps, pooled K and
every selected block id bit-exact, attention outputs within BASELINE.json's 2e-2 / 2e-3 (uf_harness.oracle_fused_step).
A separate test compares the kernel with a float32 model of itself (tests/fused_fp32_model.py): that one shows the bits
are reproducible, not that they are right."""
import numpy as np
import pytest

import uf_workloads as wl
import uf_harness as hz
from test_gpu_parity import _check_cache

pytestmark = pytest.mark.gpu


def _stream(w, n_chunks, lens=None, windows=None, fused_qkv=False, **sel):
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    rs = hz.RopeState(w, 64, cu.dev)
    try:
        for c in range(n_chunks):
            n = None if lens is None else lens[c]
            win = 0 if windows is None else windows[c]
            Qb, Kb, Vb = wl.make_chunk(w, c, n_tokens=n)
            t0 = c * w.frames_per_chunk
            got = hz.fused_step(cu, rs, Qb, Kb, Vb, t0, window=win, fused_qkv=fused_qkv, **sel)
            ref = hz.oracle_fused_step(orc, rs, w, Qb, Kb, Vb, t0, got, cu, c, window=win, **sel)
            hz.compare_step(got, ref, f"[{w.name} fused chunk {c}]")
            # fused append (1) + score / top-k / pair merge (1 kernel, no pooling pass) + attention (2); chunk 0 has no candidates
            assert got["launches"] == (4 if got["k_eff"] > 0 else 3), got["launches"]
        _check_cache(cu, orc, w)                           # cache bytes == oracle's post-RoPE K, V; pooled K bit-exact
    finally:
        cu.close()


def test_fused_small_stream_ragged():
    w = wl.scaled(wl.CONFIGS["1k"], "fz_small", n_heads=2, frames_per_chunk=2, grid_h=13, grid_w=21, capacity_chunks=3,
                  topk_percent=50)
    assert w.chunk_tokens == 546 and w.bpc == 5
    _stream(w, 5, topk_percent=50)


def test_fused_strided_qkv_variable_length_and_windows():
    """Q, K, V as slices of one [n, 3, H, d] projection output; chunks of different lengths (the last frame partial);
    shrinking windows; S = 2 sink blocks."""
    w = wl.scaled(wl.CONFIGS["1k"], "fz_var", n_heads=3, frames_per_chunk=2, grid_h=10, grid_w=20, capacity_chunks=4,
                  sink_blocks=2)
    _stream(w, 6, lens=[400, 333, 400, 129, 257, 400], windows=[0, 0, 0, 2, 4, 3], fused_qkv=True, topk_count=2)


def test_fused_error_codes():
    import torch
    import paper_2606_09150_b200 as uf
    w = wl.scaled(wl.CONFIGS["1k"], "fz_err", n_heads=1, frames_per_chunk=1, grid_h=16, grid_w=16, capacity_chunks=2)
    cu = hz.CudaStream(w)
    rs = hz.RopeState(w, 16, cu.dev)
    try:
        Qb, Kb, Vb = wl.make_chunk(w, 0)
        q, k, v = cu.to_dev(Qb), cu.to_dev(Kb), cu.to_dev(Vb)
        qo = torch.empty_like(q)
        args = (cu.ctx, q, k, v, qo, 256, 128, 128, 128, 128, rs.d_cos, rs.d_sin, rs.d_gq, rs.d_gk)
        with pytest.raises(uf.UFError) as ei:                       # t0 + frames > max_pos
            uf.uf_qkv_rope_append(*args, 16, 16, 16, 16, stream=cu.stream)
        assert ei.value.code == uf.binding.UF_ERR_CAPACITY
        with pytest.raises(uf.UFError) as ei:                       # axis dims do not sum to head_dim
            uf.uf_qkv_rope_append(*args, 16, 0, 16, 16, dims=(44, 42, 40), stream=cu.stream)
        assert ei.value.code == uf.binding.UF_ERR_INVALID_ARG
        assert uf.uf_get_slot_map(cu.ctx, 2) == ([-1, -1], 0, -1)   # nothing was appended
        uf.uf_qkv_rope_append(*args, 16, 0, 16, 16, stream=cu.stream)
        assert uf.uf_get_slot_map(cu.ctx, 2) == ([0, -1], 1, 0)
        # a select call with ANOTHER q buffer must not reuse the pooled Q of the fused call
        l0 = uf.uf_ctx_launch_count(cu.ctx)
        uf.uf_kv_append(cu.ctx, k, v, 256, 128, 128, 0, cu.stream)
        uf.uf_select_blocks(cu.ctx, q, 256, 128, 128, 1, -1, None, None, cu.stream)
        assert uf.uf_ctx_launch_count(cu.ctx) - l0 == 1 + 2         # append + pool + (score, top-k, pair merge)
        torch.cuda.synchronize()
    finally:
        cu.close()


def test_fused_full_size_1k():
    """BASELINE.json configs[1] shapes through the fused entry: all 2 x 50.1 M post-RoPE Q elements and all cached K
    within one bf16 ulp of the fp64 oracle; all selected block ids, sampled pooled K bit-exact against the oracle fed with
    the kernel's bits; attention on sampled (head, query block) pairs."""
    w = wl.CONFIGS["1k"]
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    rs = hz.RopeState(w, 128, cu.dev)
    try:
        for c in range(2):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            got = hz.fused_step(cu, rs, Qb, Kb, Vb, 3 * c, topk_percent=w.topk_percent)
            ref = hz.oracle_fused_step(orc, rs, w, Qb, Kb, Vb, 3 * c, got, cu, c, topk_percent=w.topk_percent,
                                       heads=[0, 5, 11], qblocks=[0, 1, 77, 190, 191], attn=(c == 1))
            r = hz.compare_step(got, ref, f"[1k fused chunk {c}]")
        print(f"1k fused: Q / K bit-equal to the fp64 oracle's rounding {ref['eq_q']:.5f} / {ref['eq_k']:.5f}, sampled O "
              f"max-abs {r[0]:.3e} mean-abs {r[1]:.3e}, min top-k gap {ref['min_gap']:.3e}")
        _check_cache(cu, orc, w)
    finally:
        cu.close()


def test_fused_in_place_overlap_and_rewritten_q_out():
    """(a) q_out == q_in (same strides) gives the bits of the out-of-place call, also inside a fused
    [n, 3, H, d] tensor; (b) any other overlap of q_out with an input is refused and nothing is appended; (c) a q_out
    rewritten between the fused append and the select is recognised by address only: with the shortcut on the selection
    is the one for the ORIGINAL q_out (documented), with uf_set_pooled_q_reuse(ctx, 0) it follows the q argument."""
    import torch
    import paper_2606_09150_b200 as uf
    w = wl.scaled(wl.CONFIGS["1k"], "fz_alias", n_heads=2, frames_per_chunk=2, grid_h=16, grid_w=24, capacity_chunks=3)
    n, H, d = w.chunk_tokens, 2, 128
    rs = None
    outs = {}
    for mode in ("separate", "in_place", "in_place_fused"):
        cu = hz.CudaStream(w)
        rs = rs or hz.RopeState(w, 64, cu.dev)
        try:
            for c in range(2):
                Qb, Kb, Vb = wl.make_chunk(w, c)
                if mode == "in_place_fused":
                    qkv = cu.to_dev(np.ascontiguousarray(np.stack([Qb, Kb, Vb], axis=1)))
                    q, k, v, ts = qkv[:, 0], qkv[:, 1], qkv[:, 2], 3 * H * d
                else:
                    q, k, v, ts = cu.to_dev(Qb), cu.to_dev(Kb), cu.to_dev(Vb), H * d
                q_out = torch.empty((n, H, d), dtype=torch.bfloat16, device=cu.dev) if mode == "separate" else q
                ots = H * d if mode == "separate" else ts
                uf.uf_qkv_rope_append(cu.ctx, q, k, v, q_out, n, ts, d, ots, d, rs.d_cos, rs.d_sin, rs.d_gq, rs.d_gk,
                                      rs.max_pos, 2 * c, w.grid_h, w.grid_w, wl.ROPE_AXIS_DIMS, 1e-6, 0, cu.stream)
                if mode == "in_place_fused":                      # the K and V slices are inputs only
                    torch.cuda.synchronize(cu.dev)
                    assert np.array_equal(qkv[:, 1].contiguous().view(torch.int16).cpu().numpy().view(np.uint16), Kb)
                    assert np.array_equal(qkv[:, 2].contiguous().view(torch.int16).cpu().numpy().view(np.uint16), Vb)
            _, k_eff = uf.uf_query_topk(cu.ctx, -1, 50)
            idx = torch.full((H, w.bpc, k_eff), -1, dtype=torch.int32, device=cu.dev)
            uf.uf_select_blocks(cu.ctx, q_out, n, ots, d, -1, 50, idx, None, cu.stream)
            torch.cuda.synchronize(cu.dev)
            outs[mode] = (q_out.contiguous().view(torch.int16).cpu().numpy().view(np.uint16), idx.cpu().numpy())
            if mode != "separate":
                continue
            # (c) rewrite q_out: the other chunk's raw Q, as if the caller had reused the buffer
            other = cu.to_dev(wl.make_chunk(w, 7)[0])
            backup = q_out.clone()
            q_out.copy_(other)
            idx_stale, idx_off, idx_fresh, idx_back = (torch.full_like(idx, -1) for _ in range(4))
            l0 = uf.uf_ctx_launch_count(cu.ctx)
            uf.uf_select_blocks(cu.ctx, q_out, n, H * d, d, -1, 50, idx_stale, None, cu.stream)
            assert uf.uf_ctx_launch_count(cu.ctx) - l0 == 1                 # shortcut taken: no pooling pass
            uf.uf_set_pooled_q_reuse(cu.ctx, False)
            l0 = uf.uf_ctx_launch_count(cu.ctx)
            uf.uf_select_blocks(cu.ctx, q_out, n, H * d, d, -1, 50, idx_off, None, cu.stream)
            assert uf.uf_ctx_launch_count(cu.ctx) - l0 == 2                 # pooled again
            fresh = other.clone()                              # same values at another address: always pooled
            uf.uf_select_blocks(cu.ctx, fresh, n, H * d, d, -1, 50, idx_fresh, None, cu.stream)
            # a select that pooled another Q has overwritten the ctx's pooled-Q table: with the shortcut back on, the
            # original q_out must be pooled again, not matched by address against a table that no longer holds it
            uf.uf_set_pooled_q_reuse(cu.ctx, True)
            q_out.copy_(backup)
            l0 = uf.uf_ctx_launch_count(cu.ctx)
            uf.uf_select_blocks(cu.ctx, q_out, n, H * d, d, -1, 50, idx_back, None, cu.stream)
            assert uf.uf_ctx_launch_count(cu.ctx) - l0 == 2
            torch.cuda.synchronize(cu.dev)
            assert np.array_equal(idx_stale.cpu().numpy(), outs["separate"][1])      # the documented hazard
            assert np.array_equal(idx_off.cpu().numpy(), idx_fresh.cpu().numpy())
            assert not np.array_equal(idx_fresh.cpu().numpy(), outs["separate"][1])
            assert np.array_equal(idx_back.cpu().numpy(), outs["separate"][1])
            # (b) overlaps that are refused; the ctx stays where it was
            before = uf.uf_get_slot_map(cu.ctx, w.capacity_chunks)
            flat = torch.zeros(4 * n * H * d, dtype=torch.bfloat16, device=cu.dev)
            view = lambda off: flat[off:off + n * H * d].view(n, H, d)
            a, b, cbuf = view(0), view(n * H * d), view(2 * n * H * d)
            for qo, qi, ki, vi in ((a, b, a, cbuf),                                  # q_out == k_in
                                   (view(H * d), a, b + 0, cbuf),                    # q_out = q_in shifted by one row
                                   (view(n * H * d - 8), a, view(2 * n * H * d), view(3 * n * H * d))):   # tail of q_in ... head of k_in
                with pytest.raises(uf.UFError) as ei:
                    uf.uf_qkv_rope_append(cu.ctx, qi, ki, vi, qo, n, H * d, d, H * d, d, rs.d_cos, rs.d_sin, rs.d_gq,
                                          rs.d_gk, rs.max_pos, 4, w.grid_h, w.grid_w, wl.ROPE_AXIS_DIMS, 1e-6, 0, cu.stream)
                assert ei.value.code == uf.binding.UF_ERR_INVALID_ARG
            assert uf.uf_get_slot_map(cu.ctx, w.capacity_chunks) == before
        finally:
            cu.close()
    for mode in ("in_place", "in_place_fused"):
        assert np.array_equal(outs[mode][0], outs["separate"][0]), f"{mode}: post-RoPE Q differs from the out-of-place call"
        assert np.array_equal(outs[mode][1], outs["separate"][1]), f"{mode}: selection differs"


def test_fused_bits_equal_the_float32_model_of_the_kernel():
    """Reproducibility, not correctness: the kernel's post-RoPE Q bits equal tests/fused_fp32_model.py (a NumPy
    float32 restatement of the kernel's own operation order) bit for bit, so cache bytes and block indices are a fixed
    function of the input bits on any device."""
    import fused_fp32_model as fm
    w = wl.scaled(wl.CONFIGS["1k"], "fz_model", n_heads=2, frames_per_chunk=2, grid_h=13, grid_w=21, capacity_chunks=2)
    cu = hz.CudaStream(w)
    rs = hz.RopeState(w, 64, cu.dev)
    try:
        Qb, Kb, Vb = wl.make_chunk(w, 0)
        got = hz.fused_step(cu, rs, Qb, Kb, Vb, 5, topk_count=0)
        pos = fm.raster_positions(Qb.shape[0], w.grid_h, w.grid_w, 5)
        assert np.array_equal(got["q_out_bits"], fm.apply(hz.bits_to_f64(Qb), rs.gq, rs.cos, rs.sin, pos))
        k_gpu, _ = hz.cache_chunk_bits(cu, 0, Qb.shape[0])
        assert np.array_equal(k_gpu, fm.apply(hz.bits_to_f64(Kb), rs.gk, rs.cos, rs.sin, pos))
    finally:
        cu.close()
