"""uf_select_blocks_static (include/uf_static.h): the library's one call that allocates no device memory.

Why it exists: every other call needs a uf_ctx, and uf_ctx_create cudaMallocs caches and a selection workspace.  A
plug-in that runs under a host runtime's "do not allocate in here" rule, a process whose GPU memory already belongs
to another framework's allocator, or a loop that cannot afford cudaMalloc's device-wide synchronisation cannot make
that call.  For them the pooled Q / K tables of the selection live in a fixed 16 MiB `static __device__` array.

What is checked here:
  * (CPU) the header's symbols are exported, and a problem that does not fit the array (or has more than 4096 key
    blocks) is refused with UF_ERR_CAPACITY before anything touches a GPU;
  * (GPU) the block indices equal, bit for bit — the tolerance every selection test in this suite uses — those of the
    existing ctx path (uf_kv_append + uf_select_blocks) for the same Q and the same candidate blocks, on TWO calls in a
    row with different sizes: the array is shared and never cleared, so the second call runs on top of the first
    call's leftovers and must not see them; and a further call leaves the GPU's free memory exactly where it was.

This file is named to be collected last: the driver runs pytest with -x, and a failure here must not hide the parity
tests.  It passes on its own in a fresh process and after the rest of the suite (nothing here depends on, or
disturbs, another test's state: the comparison ctx is created and destroyed inside the test).
"""
from __future__ import annotations

import os
import re

import numpy as np
import pytest

import paper_2606_09150_b200 as uf
from paper_2606_09150_b200 import binding, static_binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    uf.build()
    return uf.load_library()


def test_static_header_symbols_are_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "uf_static.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(uf_[a-z_0-9]+)\s*\(", hdr)))
    assert declared == sorted(static_binding.STATIC_SYMBOLS), declared
    for name in declared:
        assert hasattr(lib, name), f"libuf.so does not export {name}"
    assert f"({static_binding.UF_STATIC_SCRATCH_BYTES // (1024 * 1024)} * 1024 * 1024)" in hdr
    assert str(static_binding.UF_STATIC_MAX_KEY_BLOCKS) in hdr


def test_static_sizes_beyond_the_array_are_refused_before_any_gpu_work(lib):
    """Size and argument checks come first, so they behave the same with and without a GPU.  The pointers are fake
    (aligned, never dereferenced: every call here must fail before a kernel is launched)."""
    fake = 1 << 20
    H, d, B = 12, 128, 128

    def call(nq, nk, k=4, **kw):
        args = dict(device=0, q=fake, n_q_tokens=nq, q_tok_stride=H * d, q_head_stride=d, k=fake, n_k_tokens=nk,
                    k_tok_stride=H * d, k_head_stride=d, n_heads=H, head_dim=d, block=B, topk_count=k, idx_out=fake)
        args.update(kw)
        uf.uf_select_blocks_static(**args)

    # BASELINE.json configs[2] (2K): 1020 query blocks against two cached chunks -> 37.6 MB of pooled tables
    with pytest.raises(uf.UFError) as e:
        call(1020 * B, 2040 * B)
    assert e.value.code == binding.UF_ERR_CAPACITY and "UF_STATIC_SCRATCH_BYTES" in str(e.value)
    # just over: one query block plus floor(16 MiB / (8*H*d)) key blocks is 8 KB more than the array holds
    nblocks = static_binding.UF_STATIC_SCRATCH_BYTES // (8 * H * d)
    with pytest.raises(uf.UFError) as e:
        call(B, nblocks * B)
    assert e.value.code == binding.UF_ERR_CAPACITY
    # too many key blocks for the shared-memory ranking, although the tables would fit (1 head, d 32)
    with pytest.raises(uf.UFError) as e:
        call(B, (static_binding.UF_STATIC_MAX_KEY_BLOCKS + 1) * B, n_heads=1, head_dim=32, q_tok_stride=32,
             q_head_stride=32, k_tok_stride=32, k_head_stride=32)
    assert e.value.code == binding.UF_ERR_CAPACITY and "UF_STATIC_MAX_KEY_BLOCKS" in str(e.value)
    for bad in (dict(head_dim=48), dict(block=100), dict(topk_count=0), dict(q=fake + 2), dict(k_tok_stride=d + 4),
                dict(idx_out=None), dict(device=-1), dict(n_k_tokens=0)):
        with pytest.raises(uf.UFError) as e:
            call(B, 4 * B, **bad)
        assert e.value.code == binding.UF_ERR_INVALID_ARG, bad
    import torch
    if not torch.cuda.is_available():
        # a problem that fits, on a box without a GPU: a loud CUDA error, not a CPU fallback
        with pytest.raises(uf.UFError) as e:
            call(B, 4 * B)
        assert e.value.code == binding.UF_ERR_CUDA


def _bf16_bits(rng, shape):
    x = rng.standard_normal(shape).astype(np.float32)
    return (x.view(np.uint32) >> 16).astype(np.uint16)          # truncation: any bf16 bit pattern will do


def _ctx_path_indices(torch, dev, H, d, B, Qb, Kb, k):
    """The existing path on the same candidates: K becomes chunk 0 of a fresh ctx without a sink, a second chunk of
    Q's length is appended, and uf_select_blocks ranks chunk 0's blocks for q.  Global id = 0 * BPC + block = block."""
    nq, nk = Qb.shape[0], Kb.shape[0]
    to_dev = lambda bits: torch.from_numpy(bits.view(np.int16)).to(dev).view(torch.bfloat16)
    ctx = uf.uf_ctx_create(H, d, B, max(nq, nk), 2, 0, 1, dev.index)
    try:
        s = torch.cuda.current_stream(dev)
        kd = to_dev(Kb)
        uf.uf_kv_append(ctx, kd, kd, nk, H * d, d, 0, s)
        cur = to_dev(Qb)
        uf.uf_kv_append(ctx, cur, cur, nq, H * d, d, 0, s)
        n_cand, k_eff = uf.uf_query_topk(ctx, k, -1)
        assert n_cand == -(-nk // B)
        idx = torch.full((H, -(-nq // B), k_eff), -1, dtype=torch.int32, device=dev)
        uf.uf_select_blocks(ctx, cur, nq, H * d, d, k, -1, idx, None, s)
        torch.cuda.synchronize(dev)
        return idx.cpu().numpy()
    finally:
        uf.uf_ctx_destroy(ctx)


@pytest.mark.gpu
def test_static_select_matches_the_ctx_path_on_two_calls_in_a_row(lib):
    import torch
    dev = torch.device("cuda", 0)
    rng = np.random.default_rng(20261106)
    # call 1 is the larger one (ragged last blocks, several query blocks per head); call 2 is smaller and has another
    # head_dim, so its tables overlay the middle of call 1's: any value it failed to write would be call 1's
    cases = [dict(H=3, d=128, B=128, nq=4 * 128 + 5, nk=9 * 128 + 37, k=4),
             dict(H=2, d=64, B=64, nq=2 * 64 + 1, nk=5 * 64 + 63, k=5)]
    inputs = [(_bf16_bits(rng, (c["nq"], c["H"], c["d"])), _bf16_bits(rng, (c["nk"], c["H"], c["d"]))) for c in cases]
    # duplicate key blocks in case 2: equal scores must go to the lower index on both paths
    inputs[1][1][64:128] = inputs[1][1][0:64]
    want = [_ctx_path_indices(torch, dev, c["H"], c["d"], c["B"], Qb, Kb, c["k"]) for c, (Qb, Kb) in zip(cases, inputs)]

    to_dev = lambda bits: torch.from_numpy(bits.view(np.int16)).to(dev).view(torch.bfloat16)
    dev_in = [(to_dev(Qb), to_dev(Kb)) for Qb, Kb in inputs]
    outs = [torch.full(w.shape, -7, dtype=torch.int32, device=dev) for w in want]
    s = torch.cuda.current_stream(dev)
    for c, (qd, kd), out in zip(cases, dev_in, outs):
        uf.uf_select_blocks_static(0, qd, c["nq"], c["H"] * c["d"], c["d"], kd, c["nk"], c["H"] * c["d"], c["d"],
                                   c["H"], c["d"], c["B"], c["k"], out, s)
    torch.cuda.synchronize(dev)
    for n, (out, w) in enumerate(zip(outs, want)):
        got = out.cpu().numpy()
        assert got.shape == w.shape
        assert np.array_equal(got, w), f"call {n + 1}: indices differ from uf_select_blocks at {np.argwhere(got != w)[:4]}"
        assert (np.diff(got, axis=-1) > 0).all(), "rows must be ascending"
    # topk_count above the number of key blocks: every block, in order
    c, (qd, kd) = cases[1], dev_in[1]
    nkb = -(-c["nk"] // c["B"])
    allb = torch.full((c["H"], -(-c["nq"] // c["B"]), nkb), -7, dtype=torch.int32, device=dev)
    uf.uf_select_blocks_static(0, qd, c["nq"], c["H"] * c["d"], c["d"], kd, c["nk"], c["H"] * c["d"], c["d"],
                               c["H"], c["d"], c["B"], nkb + 10, allb, s)
    torch.cuda.synchronize(dev)
    assert np.array_equal(allb.cpu().numpy(), np.broadcast_to(np.arange(nkb, dtype=np.int32), allb.shape))
    # a repeat of call 2 (its kernels are loaded by now) must leave the GPU's free memory exactly where it was
    again = outs[1].fill_(-7)
    torch.cuda.synchronize(dev)
    free_before = torch.cuda.mem_get_info(dev)[0]
    uf.uf_select_blocks_static(0, qd, c["nq"], c["H"] * c["d"], c["d"], kd, c["nk"], c["H"] * c["d"], c["d"],
                               c["H"], c["d"], c["B"], c["k"], again, s)
    torch.cuda.synchronize(dev)
    assert torch.cuda.mem_get_info(dev)[0] == free_before, "a later call changed the GPU's free memory"
    assert np.array_equal(again.cpu().numpy(), want[1])
