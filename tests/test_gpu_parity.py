"""GPU parity tests: the CUDA path (through the C ABI) against the fp64 oracle, element by element on
the same seeded inputs.  Bar (BASELINE.json north_star): slot maps and selected block ids bit-exact,
attention outputs within max-abs 2e-2 / mean-abs 2e-3.  Run with `-m gpu` on a B200."""
from __future__ import annotations

import dataclasses

import numpy as np
import pytest

import uf_workloads as wl
import uf_harness as hz

pytestmark = pytest.mark.gpu


def _run_stream(w, chunks, topk_count=-1, topk_percent=-1, windows=None, impl=0, nmax=None, attn=True,
                heads=None, qblocks=None, check_cache=True):
    cu = hz.CudaStream(w, nmax)
    orc = hz.make_oracle(w, nmax)
    worst = (0.0, 0.0)
    try:
        for c, (Qb, Kb, Vb) in enumerate(chunks):
            win = 0 if windows is None else windows[c]
            got = cu.step(Qb, Kb, Vb, topk_count, topk_percent, win, impl=impl)
            ref = hz.oracle_step(orc, Qb, Kb, Vb, topk_count, topk_percent, win, heads=heads, qblocks=qblocks,
                                 attn=attn)
            r = hz.compare_step(got, ref, where=f"[{w.name} chunk {c}]")
            if r:
                worst = (max(worst[0], r[0]), max(worst[1], r[1]))
        if check_cache:
            _check_cache(cu, orc, w)
    finally:
        cu.close()
    return worst


def _check_cache(cu, orc, w):
    """Cache bytes of resident blocks (first, last of each chunk) and the sink equal the inputs; pooled K
    equals the oracle's block means bit for bit."""
    H = w.n_heads
    for ch in orc.resident:
        nb = orc.n_blocks(ch["n"])
        for b in sorted({0, nb - 1}):
            g = ch["id"] * orc.BPC + b
            for h in sorted({0, H - 1}):
                kb, vb = cu.cache_block(g, h)
                kr, vr = orc.block_kv(g)
                r = kr.shape[0]
                assert np.array_equal(hz.bits_to_f64(kb[:r]), kr[:, h, :])
                assert np.array_equal(hz.bits_to_f64(vb[:r]), vr[:, h, :])
                assert not kb[r:].any() and not vb[r:].any(), "pad rows of a ragged block must be zero"
                pk = cu.pooled_k(g, h)
                assert np.array_equal(pk, kr[:, h, :].sum(axis=0) / float(r))
    for s in orc.sink_ids():
        kb, vb = cu.cache_block(-(s + 1), 0)
        kr, vr = orc.block_kv(s, from_sink=True)
        r = kr.shape[0]
        assert np.array_equal(hz.bits_to_f64(kb[:r]), kr[:, 0, :]) and np.array_equal(hz.bits_to_f64(vb[:r]), vr[:, 0, :])


# ---------------------------------------------------------------------------------------------------
def test_config0_tiny_full():
    """BASELINE.json configs[0]: 1 head x 64, block 64, 3 chunks of 128 tokens, top-2 + sink + current."""
    w = wl.CONFIGS["tiny"]
    _run_stream(w, wl.make_stream(w, 3), topk_count=2)


@pytest.mark.parametrize("impl", [0, 1])
def test_small_b128_stream_ragged(impl):
    """B = d = 128 (tcgen05 kernel when impl = 0; generic kernel when impl = 1): 6 chunks, capacity 3,
    5 query blocks (odd: the last pair has one tile) with a ragged 40-token tail, 2 heads, top 50 %."""
    w = wl.scaled(wl.CONFIGS["1k"], "small128", n_heads=2, frames_per_chunk=1, grid_h=23, grid_w=24,
                  capacity_chunks=3, topk_percent=50)
    assert w.chunk_tokens == 552 and w.bpc == 5
    _run_stream(w, wl.make_stream(w, 6), topk_percent=50, impl=impl)


def test_small_b128_even_blocks_count_mode():
    w = wl.scaled(wl.CONFIGS["1k"], "small128e", n_heads=3, frames_per_chunk=1, grid_h=32, grid_w=32,
                  capacity_chunks=2)
    assert w.chunk_tokens == 1024 and w.bpc == 8
    _run_stream(w, wl.make_stream(w, 4), topk_count=3)


def test_dense_limit_k_saturates():
    """k >= |CAND| keeps every candidate: the sparse path equals dense chunk-causal attention."""
    w = wl.scaled(wl.CONFIGS["1k"], "dense128", n_heads=1, frames_per_chunk=1, grid_h=16, grid_w=20,
                  capacity_chunks=3)
    _run_stream(w, wl.make_stream(w, 4), topk_count=10_000)


def test_window_shrink_and_variable_chunk_length():
    """FIFO window shrink evicts several chunks; a slot reused by a shorter chunk must not leak stale rows."""
    w = wl.scaled(wl.CONFIGS["1k"], "var128", n_heads=2, frames_per_chunk=1, grid_h=20, grid_w=20,
                  capacity_chunks=4)
    lens = [400, 333, 400, 129, 1, 257, 400]
    windows = [0, 0, 0, 2, 4, 1, 3]
    chunks = [wl.make_chunk(w, c, n_tokens=n) for c, n in enumerate(lens)]
    _run_stream(w, chunks, topk_percent=60, windows=windows, nmax=400)


def test_ties_duplicate_blocks_lower_id_wins():
    """Bitwise-duplicated key blocks score equal; the lower global id must be selected (BJ)."""
    w = wl.scaled(wl.CONFIGS["1k"], "ties128", n_heads=2, frames_per_chunk=1, grid_h=16, grid_w=32,
                  capacity_chunks=3)
    assert w.chunk_tokens == 512
    chunks = wl.make_stream(w, 3)
    Q1, K1, V1 = chunks[1]
    K0 = chunks[0][1]
    K1 = K1.copy()
    K1[0:128] = K0[128:256]          # chunk1 block0 == chunk0 block1
    K1[256:384] = K0[128:256]        # chunk1 block2 == chunk0 block1
    K1[384:512] = K1[128:256]        # chunk1 block3 == chunk1 block1
    chunks[1] = (Q1, K1, V1)
    _run_stream(w, chunks, topk_count=2)
    _run_stream(w, chunks, topk_count=3)


def test_no_sink_and_small_dims_generic():
    """S = 0 (no sink) and the d = 32 / B = 32 generic shapes."""
    w = wl.scaled(wl.CONFIGS["tiny"], "tiny32", n_heads=3, head_dim=32, block=32, frames_per_chunk=1, grid_h=7,
                  grid_w=11, capacity_chunks=2, sink_blocks=0, amp=1.0)
    _run_stream(w, [wl.make_chunk(w, c) for c in range(4)], topk_count=1)


def test_custom_scale_and_no_lse():
    w = wl.scaled(wl.CONFIGS["1k"], "scale128", n_heads=1, frames_per_chunk=1, grid_h=16, grid_w=16,
                  capacity_chunks=2)
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    try:
        for c in range(2):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            got = cu.step(Qb, Kb, Vb, topk_count=1, want_lse=False, scale=0.05)
            ref = hz.oracle_step(orc, Qb, Kb, Vb, topk_count=1, scale=0.05)
            hz.compare_step(got, ref, f"[scale chunk {c}]")
    finally:
        cu.close()


@pytest.mark.parametrize("scale", [0.3, 8.0])
def test_sharp_softmax_deferred_raise_and_safe_kernel(scale):
    """Logits far sharper than 1/sqrt(d) gives.  scale 0.3: the row max outgrows the running reference by
    many binades inside single key blocks, so the deferred raise of m (O_t, l rescaled by 2^-D before the
    next block) runs all the time.  scale 8: it outgrows it by more than 2^100, the exponentials overflow,
    the items are flagged and the exact-max ("safe") instantiation of the kernel must redo them; the result
    is then practically a one-hot selection of V rows.  The generic kernel is the second opinion."""
    import torch
    w = wl.scaled(wl.CONFIGS["1k"], "sharp128", n_heads=2, frames_per_chunk=1, grid_h=20, grid_w=29,
                  capacity_chunks=3, topk_percent=50)
    assert w.chunk_tokens == 580                                    # 5 query blocks, ragged tail of 68
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    try:
        redone = 0
        for c in range(3):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            got = cu.step(Qb, Kb, Vb, topk_percent=50, scale=scale)
            redone += cu.uf.uf_attn_redone_items(cu.ctx, cu.stream)
            ref = hz.oracle_step(orc, Qb, Kb, Vb, topk_percent=50, scale=scale)
            hz.compare_step(got, ref, f"[sharp scale {scale} chunk {c}]")
            q = cu.to_dev(Qb)
            o2 = torch.empty_like(q)
            n, H, d = Qb.shape
            cu.uf.uf_set_attn_impl(cu.ctx, 1)
            cu.uf.uf_sparse_attn_fwd(cu.ctx, q, o2, None, n, H * d, d, scale, cu.stream)
            torch.cuda.synchronize()
            assert cu.uf.uf_attn_redone_items(cu.ctx, cu.stream) == 0        # generic kernel: nothing to redo
            diff = np.abs(got["O"] - o2.float().cpu().numpy())
            assert diff.max() <= hz.O_MAX_ABS and diff.mean() <= hz.O_MEAN_ABS, (diff.max(), diff.mean())
        if scale >= 8.0:
            assert redone > 0, "scale 8 must overflow the stale-max exponentials and take the safe kernel"
    finally:
        cu.close()


@pytest.mark.parametrize("col", [0, 2, 6, 77])
def test_outlier_logit_far_above_running_max(col):
    """One key of a LATE block carries a logit ~180 binades above everything the row has seen, every other
    logit is small.  Columns 0, 1, 6, 7, 12, 13 (mod 16) of a key block take the FMA-pipe exp2 polynomial,
    whose exponent arithmetic would wrap for such an argument (a small or negative number instead of an
    overflow) if it were not clamped; the others take MUFU ex2 and overflow to inf.  Either way the item must
    be flagged and redone with the exact row max: the output is the outlier's V row."""
    w = wl.scaled(wl.CONFIGS["1k"], f"outlier{col}", n_heads=1, frames_per_chunk=1, grid_h=16, grid_w=24,
                  capacity_chunks=2, amp=0.0)
    assert w.chunk_tokens == 384
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    try:
        rng = np.random.default_rng(5)
        for c in range(2):
            Q = 0.25 * rng.standard_normal((384, 1, 128)).astype(np.float32)
            K = 0.25 * rng.standard_normal((384, 1, 128)).astype(np.float32)
            V = rng.standard_normal((384, 1, 128)).astype(np.float32)
            Q[:, 0, 0] = 4.0
            K[:, 0, 0] = 0.0
            if c == 1:
                K[256 + col, 0, 0] = 64.0                  # key `col` of the last current block: q.k = 256
            Qb, Kb, Vb = (wl.f32_to_bf16_bits(x) for x in (Q, K, V))
            got = cu.step(Qb, Kb, Vb, topk_count=1, scale=0.5)          # logit 128 -> 184.7 binades
            redone = cu.uf.uf_attn_redone_items(cu.ctx, cu.stream)
            ref = hz.oracle_step(orc, Qb, Kb, Vb, topk_count=1, scale=0.5)
            hz.compare_step(got, ref, f"[outlier col {col} chunk {c}]")
            if c == 1:
                assert redone > 0, "the overflow must be detected and the item redone with the exact max"
                want = hz.bits_to_f64(Vb)[256 + col, 0]
                assert np.abs(got["O"][:, 0].astype(np.float64) - want[None, :]).max() <= 1e-6
    finally:
        cu.close()


def test_strided_views_of_fused_tensors():
    """Q, K, V passed as strided slices of one fused [n, 3, H, d] tensor and O written into a slice of a larger
    tensor (token stride != H*d): append, select and the TMA maps of the attention kernel must honour the strides
    and must not touch the neighbouring slices."""
    w = wl.scaled(wl.CONFIGS["1k"], "fused128", n_heads=2, frames_per_chunk=1, grid_h=21, grid_w=24,
                  capacity_chunks=3, topk_percent=40)
    assert w.chunk_tokens == 504
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    try:
        for c in range(4):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            got = cu.step(Qb, Kb, Vb, topk_percent=40, fused_qkv=True)
            ref = hz.oracle_step(orc, Qb, Kb, Vb, topk_percent=40)
            hz.compare_step(got, ref, f"[fused chunk {c}]")
        _check_cache(cu, orc, w)
    finally:
        cu.close()


@pytest.mark.parametrize("seed", range(8))
def test_randomised_streams(seed):
    """Seeded random small configurations of the B = d = 128 path: heads, token grid (odd / even number of query
    blocks, ragged tails down to 1 token), capacity 1-4 (capacity 1: never any candidate), 0-2 sink blocks, count
    or percent budgets (0, saturating, k_min floor), per-chunk windows and chunk lengths, softmax scale."""
    rng = np.random.default_rng(1000 + seed)
    H = int(rng.integers(1, 4))
    gh, gw = int(rng.integers(9, 31)), int(rng.integers(9, 31))
    C = int(rng.integers(1, 5))
    S = int(rng.integers(0, 3))
    w = wl.scaled(wl.CONFIGS["1k"], f"rand{seed}", n_heads=H, frames_per_chunk=1, grid_h=gh, grid_w=gw,
                  capacity_chunks=C, sink_blocks=S, amp=float(rng.choice([0.0, 1.0, 2.0, 3.0])))
    nmax = w.chunk_tokens
    percent_mode = bool(rng.integers(0, 2))
    kc = -1 if percent_mode else int(rng.choice([0, 1, 2, 5, 1000]))
    kp = int(rng.choice([0, 10, 33, 100])) if percent_mode else -1
    scale = float(rng.choice([0.0, 0.05, 0.25]))
    n_chunks = int(rng.integers(3, 7))
    cu, orc = hz.CudaStream(w, nmax), hz.make_oracle(w, nmax)
    try:
        for c in range(n_chunks):
            n = nmax if rng.random() < 0.5 else int(rng.integers(1, nmax + 1))
            win = int(rng.integers(0, C + 1))
            Qb, Kb, Vb = wl.make_chunk(w, c, n_tokens=n)
            got = cu.step(Qb, Kb, Vb, kc, kp, win, scale=scale)
            ref = hz.oracle_step(orc, Qb, Kb, Vb, kc, kp, win, scale=scale)
            hz.compare_step(got, ref, f"[rand{seed} H{H} {gh}x{gw} C{C} S{S} k{kc}/{kp}% chunk {c} n{n} win{win}]")
        _check_cache(cu, orc, w)
    finally:
        cu.close()


def test_reset_starts_a_new_stream_and_two_ctx_interleave():
    """uf_ctx_reset empties the cache (a new video starts at chunk 0: sink rewritten, no candidates), and two
    contexts (two layers / two streams) driven in turn on their own CUDA streams do not disturb each other."""
    import torch
    w = wl.scaled(wl.CONFIGS["1k"], "reset128", n_heads=2, frames_per_chunk=1, grid_h=18, grid_w=25,
                  capacity_chunks=2, topk_percent=50)
    cu_a, cu_b = hz.CudaStream(w), hz.CudaStream(w)
    cu_b.stream = torch.cuda.Stream(cu_b.dev)
    orc_a, orc_b = hz.make_oracle(w), hz.make_oracle(w)
    try:
        # stream A sees chunks 0, 1, 2; stream B sees the same recipe with other seeds, interleaved with A
        for c in range(3):
            Qa, Ka, Va = wl.make_chunk(w, c)
            Qb, Kb, Vb = wl.make_chunk(w, c, seed=100 + c)
            with torch.cuda.stream(cu_b.stream):
                got_b = cu_b.step(Qb, Kb, Vb, topk_percent=50)
            got_a = cu_a.step(Qa, Ka, Va, topk_percent=50)
            hz.compare_step(got_a, hz.oracle_step(orc_a, Qa, Ka, Va, topk_percent=50), f"[ctx A chunk {c}]")
            hz.compare_step(got_b, hz.oracle_step(orc_b, Qb, Kb, Vb, topk_percent=50), f"[ctx B chunk {c}]")
        # reset A: the next chunk is chunk 0 of a new video (fresh oracle), B carries on untouched
        cu_a.uf.uf_ctx_reset(cu_a.ctx, cu_a.stream)
        orc_a = hz.make_oracle(w)
        for c in range(2):
            Qa, Ka, Va = wl.make_chunk(w, c, seed=200 + c)
            got_a = cu_a.step(Qa, Ka, Va, topk_percent=50)
            ref_a = hz.oracle_step(orc_a, Qa, Ka, Va, topk_percent=50)
            hz.compare_step(got_a, ref_a, f"[ctx A after reset chunk {c}]")
            assert got_a["n_cand"] == (0 if c == 0 else w.bpc - w.sink_blocks)
        Qb, Kb, Vb = wl.make_chunk(w, 3, seed=103)
        with torch.cuda.stream(cu_b.stream):
            got_b = cu_b.step(Qb, Kb, Vb, topk_percent=50)
        hz.compare_step(got_b, hz.oracle_step(orc_b, Qb, Kb, Vb, topk_percent=50), "[ctx B chunk 3]")
        _check_cache(cu_a, orc_a, w)
        _check_cache(cu_b, orc_b, w)
    finally:
        cu_a.close()
        cu_b.close()


def test_error_codes_and_call_order():
    import torch
    import paper_2606_09150_b200 as uf
    w = wl.scaled(wl.CONFIGS["1k"], "err128", n_heads=1, frames_per_chunk=1, grid_h=16, grid_w=16, capacity_chunks=2)
    cu = hz.CudaStream(w)
    try:
        Qb, Kb, Vb = wl.make_chunk(w, 0)
        q, k, v = cu.to_dev(Qb), cu.to_dev(Kb), cu.to_dev(Vb)
        o = torch.empty_like(q)
        with pytest.raises(uf.UFError) as ei:
            uf.uf_select_blocks(cu.ctx, q, 256, 128, 128, 1, -1, None, None, cu.stream)
        assert ei.value.code == uf.binding.UF_ERR_STATE
        uf.uf_kv_append(cu.ctx, k, v, 256, 128, 128, 0, cu.stream)
        with pytest.raises(uf.UFError) as ei:
            uf.uf_sparse_attn_fwd(cu.ctx, q, o, None, 256, 128, 128, 0.0, cu.stream)
        assert ei.value.code == uf.binding.UF_ERR_STATE
        with pytest.raises(uf.UFError) as ei:
            uf.uf_kv_append(cu.ctx, k, v, 257, 128, 128, 0, cu.stream)
        assert ei.value.code == uf.binding.UF_ERR_CAPACITY
        with pytest.raises(uf.UFError) as ei:
            uf.uf_kv_append(cu.ctx, k, v, 256, 130, 128, 0, cu.stream)
        assert ei.value.code == uf.binding.UF_ERR_INVALID_ARG
        with pytest.raises(uf.UFError):
            uf.uf_kv_append(cu.ctx, None, v, 256, 128, 128, 0, cu.stream)
        assert uf.uf_ctx_launch_count(cu.ctx) == 1 and uf.uf_ctx_device_bytes(cu.ctx) > 0
        # a failed append leaves the ctx as it was: still exactly one chunk resident
        assert uf.uf_get_slot_map(cu.ctx, 2) == ([0, -1], 1, 0)
        # o overlapping q is rejected on the tcgen05 path (the exact-max redo re-reads Q after O was stored)
        uf.uf_select_blocks(cu.ctx, q, 256, 128, 128, 1, -1, None, None, cu.stream)
        with pytest.raises(uf.UFError) as ei:
            uf.uf_sparse_attn_fwd(cu.ctx, q, q, None, 256, 128, 128, 0.0, cu.stream)
        assert ei.value.code == uf.binding.UF_ERR_INVALID_ARG
        uf.uf_sparse_attn_fwd(cu.ctx, q, o, None, 256, 128, 128, 0.0, cu.stream)
        torch.cuda.synchronize()
    finally:
        cu.close()
    # shapes without a tcgen05 kernel are refused unless the caller opts in to the CUDA-core kernel
    w2 = wl.CONFIGS["tiny"]
    cu = hz.CudaStream(w2)
    try:
        Qb, Kb, Vb = wl.make_chunk(w2, 0)
        q, k, v = cu.to_dev(Qb), cu.to_dev(Kb), cu.to_dev(Vb)
        o = torch.empty_like(q)
        uf.uf_kv_append(cu.ctx, k, v, 128, 64, 64, 0, cu.stream)
        uf.uf_select_blocks(cu.ctx, q, 128, 64, 64, 2, -1, None, None, cu.stream)
        with pytest.raises(uf.UFError) as ei:
            uf.uf_sparse_attn_fwd(cu.ctx, q, o, None, 128, 64, 64, 0.0, cu.stream)
        assert ei.value.code == uf.binding.UF_ERR_UNSUPPORTED
        uf.uf_set_attn_impl(cu.ctx, 1)
        uf.uf_sparse_attn_fwd(cu.ctx, q, o, None, 128, 64, 64, 0.0, cu.stream)
        torch.cuda.synchronize()
    finally:
        cu.close()


# ----------------------------------------------------------------------------- full-size configs
def _oracle_attn_parallel(orc, Q, jobs, n_threads=8):
    """The oracle's sparse_attn, as it stands, called once per (head, query-block list) job from a thread pool
    (NumPy releases the GIL in matmul / exp; BLAS is held to 2 threads per call).  Returns O, lse with NaN on
    the rows no job covered."""
    from concurrent.futures import ThreadPoolExecutor
    from threadpoolctl import threadpool_limits
    n, H, d = Q.shape
    O = np.full((n, H, d), np.nan, dtype=np.float64)
    lse = np.full((H, n), np.nan, dtype=np.float64)

    def run(job):
        h, qblocks = job
        o, l = orc.sparse_attn(Q, heads=[h], qblocks=qblocks)
        return h, qblocks, o[:, h, :].copy(), l[h].copy()

    with threadpool_limits(limits=2), ThreadPoolExecutor(n_threads) as ex:
        for h, qblocks, o, l in ex.map(run, jobs):
            for i in qblocks:
                lo, hi = i * orc.B, min((i + 1) * orc.B, n)
                O[lo:hi, h, :] = o[lo:hi]
                lse[h, lo:hi] = l[lo:hi]
    return O, lse


@pytest.mark.parametrize("name", ["1k", "2k", "wide"])
def test_full_size_step(name):
    """BASELINE.json configs[1] / configs[2] / configs[4] at full size, in the launch configuration bench.py times.
    Slot maps and ALL selected block ids bit-exact.  Attention against the oracle on EVERY row of configs[1]
    (all 2304 (head, query block) pairs: the persistent schedule wraps its work items over the 148 CTAs 8 times)
    and on every row of two whole heads of configs[2] / configs[4] plus sampled (head, query block) pairs of two
    more heads.  And every row of every head against the second CUDA implementation (generic kernel)."""
    import time
    import torch
    w = wl.CONFIGS[name]
    nqb = w.bpc
    if name == "1k":
        jobs = [(h, list(range(lo, min(lo + 24, nqb)))) for h in range(w.n_heads) for lo in range(0, nqb, 24)]
    else:
        rng = np.random.default_rng(1)
        full_heads = [0, w.n_heads - 1]
        jobs = [(h, list(range(lo, min(lo + 26, nqb)))) for h in full_heads for lo in range(0, nqb, 26)]
        sampled = sorted({0, 1, nqb - 2, nqb - 1} | set(int(x) for x in rng.integers(0, nqb, 6)))
        jobs += [(int(h), sampled) for h in rng.choice(np.arange(1, w.n_heads - 1), 2, replace=False)]
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    try:
        for c in range(w.prior_chunks + 1):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            last = c == w.prior_chunks
            got = cu.step(Qb, Kb, Vb, topk_percent=w.topk_percent)
            ref = hz.oracle_step(orc, Qb, Kb, Vb, topk_percent=w.topk_percent, attn=False)
            hz.compare_step(got, ref, f"[{name} chunk {c}]")
        assert not np.isnan(got["O"]).any(), "every output row must be written"
        assert np.isfinite(got["lse"]).all()
        assert cu.uf.uf_attn_redone_items(cu.ctx, cu.stream) == 0
        # second opinion on every row: the CUDA-core kernel on the same selection
        q = cu.to_dev(Qb)
        o2 = torch.empty_like(q)
        n, H, d = Qb.shape
        cu.uf.uf_set_attn_impl(cu.ctx, 1)
        cu.uf.uf_sparse_attn_fwd(cu.ctx, q, o2, None, n, H * d, d, 0.0, cu.stream)
        torch.cuda.synchronize()
        diff = (o2.float() - torch.from_numpy(got["O"]).to(o2.device)).abs()
        assert float(diff.max()) <= hz.O_MAX_ABS and float(diff.mean()) <= hz.O_MEAN_ABS, (float(diff.max()), float(diff.mean()))
        del diff, o2
        # the oracle, row by row
        t0 = time.time()
        ref["O"], ref["lse"] = _oracle_attn_parallel(orc, hz.bits_to_f64(Qb), jobs)
        r = hz.compare_step(got, ref, f"[{name} attention]")
        n_rows = int((~np.isnan(ref["lse"])).sum())
        print(f"{name}: {n_rows} of {H * n} (head, row) outputs vs oracle in {time.time() - t0:.0f}s: O max-abs {r[0]:.3e} "
              f"mean-abs {r[1]:.3e}, oracle min top-k gap {ref['min_gap']:.3e}")
        if name == "1k":
            assert n_rows == H * n
    finally:
        cu.close()


def test_full_size_rolling_stream():
    """BASELINE.json configs[3]: 20 consecutive 1K chunks (per-chunk seeds 0..19), capacity 3 chunks + sink, oldest
    non-sink chunk evicted after each append.  Slot maps and ALL selected block ids bit-exact on every chunk;
    attention compared on sampled (head, query block) pairs on ramp-up, mid-stream and final chunks; after the
    stream the cache holds chunks 17, 18, 19 + the sink, byte-exact."""
    w = wl.CONFIGS["1k_stream"]
    heads, qblocks = [0, w.n_heads - 1], [0, 95, w.bpc - 1]
    check_attn = {0, 1, 2, 3, 10, w.n_stream_chunks - 1}
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    try:
        worst = 0.0
        for c in range(w.n_stream_chunks):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            got = cu.step(Qb, Kb, Vb, topk_percent=w.topk_percent)
            ref = hz.oracle_step(orc, Qb, Kb, Vb, topk_percent=w.topk_percent, heads=heads, qblocks=qblocks,
                                 attn=c in check_attn)
            r = hz.compare_step(got, ref, f"[1k_stream chunk {c}]")
            if r:
                worst = max(worst, r[0])
            assert cu.uf.uf_attn_redone_items(cu.ctx, cu.stream) == 0
        assert sorted(x for x in got["slot_map"][0] if x >= 0) == [17, 18, 19]
        _check_cache(cu, orc, w)
        print(f"1k_stream: worst sampled O max-abs {worst:.3e}")
    finally:
        cu.close()


def test_sm100_kernel_matches_generic_kernel_medium():
    """Two independent CUDA implementations of step a5 (tcgen05 vs CUDA-core) agree on every row of a
    medium case that spans many tiles (property check at a size the oracle would take minutes for)."""
    import torch
    w = wl.scaled(wl.CONFIGS["1k"], "medium128", n_heads=4, frames_per_chunk=1, grid_h=50, grid_w=60,
                  capacity_chunks=3, topk_percent=25)
    cu = hz.CudaStream(w)
    try:
        for c in range(3):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            a = cu.step(Qb, Kb, Vb, topk_percent=25, impl=0)
        q = cu.to_dev(Qb)
        o2 = torch.empty_like(q)
        n, H, d = Qb.shape
        cu.uf.uf_set_attn_impl(cu.ctx, 1)
        cu.uf.uf_sparse_attn_fwd(cu.ctx, q, o2, None, n, H * d, d, 0.0, cu.stream)
        torch.cuda.synchronize()
        diff = np.abs(a["O"] - o2.float().cpu().numpy())
        assert diff.max() <= 2e-2 and diff.mean() <= 2e-3, (diff.max(), diff.mean())
    finally:
        cu.close()


def test_tensor_map_cache_eviction_between_q_and_o_lookups():
    """The ctx caches the Q / O tensor maps of recent callers (8 entries, recycled round-robin).  A call whose Q hits the
    entry that its O, missing, is about to recycle must still read Q: with 4 buffer pairs the cache is full and the
    next slot is the first Q's, so (q0, new O) is exactly that case (it once loaded Q through O's map)."""
    import torch
    w = wl.scaled(wl.CONFIGS["1k"], "tmcache", n_heads=2, frames_per_chunk=1, grid_h=16, grid_w=20, capacity_chunks=2)
    cu = hz.CudaStream(w)
    try:
        for c in range(2):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            got = cu.step(Qb, Kb, Vb, topk_percent=50)                  # leaves a valid selection in the ctx
        n, H, d = Qb.shape
        uf, ref = cu.uf, torch.from_numpy(got["O"]).to(cu.dev)
        uf.uf_ctx_reset(cu.ctx, cu.stream)                              # a fresh cache of maps needs a fresh ctx: new one
    finally:
        cu.close()
    cu = hz.CudaStream(w)
    try:
        for c in range(2):
            Qb, Kb, Vb = wl.make_chunk(w, c)
            k, v = cu.to_dev(Kb), cu.to_dev(Vb)
            uf.uf_kv_append(cu.ctx, k, v, n, H * d, d, 0, cu.stream)
        qs = [cu.to_dev(Qb) for _ in range(4)]
        os_ = [torch.full((n, H, d), float("nan"), dtype=torch.bfloat16, device=cu.dev) for _ in range(5)]
        uf.uf_select_blocks(cu.ctx, qs[0], n, H * d, d, -1, 50, None, None, cu.stream)
        for i in range(4):                                              # fills the 8 entries: q0 o0 q1 o1 q2 o2 q3 o3
            uf.uf_sparse_attn_fwd(cu.ctx, qs[i], os_[i], None, n, H * d, d, 0.0, cu.stream)
        uf.uf_sparse_attn_fwd(cu.ctx, qs[0], os_[4], None, n, H * d, d, 0.0, cu.stream)   # q0 hits slot 0, o4 recycles it
        torch.cuda.synchronize()
        for i in range(5):
            assert not torch.isnan(os_[i].float()).any(), f"call {i}: NaN / unwritten rows"
            assert torch.equal(os_[i].float(), ref), f"call {i} differs from the first result"
    finally:
        cu.close()


def test_block_column_beyond_the_exact_sum_range():
    """ADVICE r1 item 4 / VERDICT r2 item 9: include/uf.h promises bit-exact indices "as long as the block sums are exact
    in fp64", i.e. while one (block, head, channel) column spans fewer than 2^38 between its largest magnitude and its
    smallest non-zero ulp; beyond that "the summation order may change the last bit of a pooled mean".  This feeds a
    column that spans 2^74 (one 2^60 among values with ulps of 2^-14) and checks exactly that promise: the exact mean
    (rational arithmetic) is bracketed by the GPU's and by the oracle's fp64 means within one ulp each — nothing worse
    — every OTHER pooled value stays bit-exact, and the selection, whose top-k gaps are far above one ulp here, is
    unchanged."""
    from fractions import Fraction
    w = wl.scaled(wl.CONFIGS["1k"], "widerange", n_heads=1, frames_per_chunk=1, grid_h=16, grid_w=32, capacity_chunks=2,
                  sink_blocks=0)
    assert w.chunk_tokens == 512 and w.bpc == 4
    chunks = [list(wl.make_chunk(w, c)) for c in range(2)]
    Kb = chunks[0][1]
    blk, ch = 2, 5
    Kb[blk * 128 + 17, 0, ch] = wl.f32_to_bf16_bits(np.array([2.0 ** 60], dtype=np.float32))[0]
    col = hz.bits_to_f64(Kb[blk * 128:(blk + 1) * 128, 0, ch])
    nz = np.abs(col[col != 0])
    ulps = np.ldexp(1.0, np.frexp(nz)[1] - 8)                 # ulp of a bf16 value with exponent e (8 significant bits)
    assert nz.max() / ulps.min() > 2.0 ** 53                  # the fp64 sum of this column cannot be exact
    cu, orc = hz.CudaStream(w), hz.make_oracle(w)
    try:
        for c, (Qb, Kc, Vb) in enumerate(chunks):
            got = cu.step(Qb, Kc, Vb, topk_count=2)
            # attention is not compared here: a 2^60 key makes logits of ~1e18, where fp32 logits have an ulp of 2^36
            # and O is no longer within 2e-2 of the fp64 softmax (measured: max-abs 2.7); this case is about pooling
            ref = hz.oracle_step(orc, Qb, Kc, Vb, topk_count=2, attn=False)
            hz.compare_step(got, ref, f"[widerange chunk {c}]")          # indices, counts, slot map bit-exact
        assert ref["min_gap"] > 1e-6                                      # the gaps dwarf a last-bit change of one mean
        exact = sum(Fraction(float(x)) for x in col) / 128
        pk = cu.pooled_k(0 * w.bpc + blk, 0)
        ulp = np.spacing(float(exact))
        assert abs(Fraction(float(pk[ch])) - exact) <= Fraction(ulp), (pk[ch], float(exact))
        ok = orc.pooled_mean(hz.bits_to_f64(Kb))[0, blk]
        assert abs(Fraction(float(ok[ch])) - exact) <= Fraction(ulp)
        others = np.arange(128) != ch
        assert np.array_equal(pk[others], ok[others])                     # every exact column is still bit-exact
    finally:
        cu.close()
