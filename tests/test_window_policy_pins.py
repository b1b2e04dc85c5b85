"""Pins of the window-policy oracle (oracle/uf_window_policy.py, NEXT-3) and, through a host-only ctx, of the C ABI's
uf_next_window for the two policies that need no device (position, memory).  CPU only."""
import numpy as np
import pytest

import uf_workloads as wl
from oracle import UFOracle
from oracle import uf_window_policy as wp


def bf16(x):
    return wl.bf16_bits_to_f32(wl.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))).astype(np.float64)


def chunk(rng, n, H, d, kscale=1.0):
    Q, K, V = (bf16(rng.standard_normal((n, H, d))) for _ in range(3))
    return Q, bf16(K * kscale), V


def test_position_policy_closed_form_and_resident_set():
    """W(c) = C for c < warm, compact afterwards; the resident set after every append is the last min(c+1, W(c)) ids."""
    rng = np.random.default_rng(0)
    C, warm, compact = 4, 6, 2
    o = UFOracle(1, 4, 4, 8, C)
    for c in range(14):
        W = wp.next_window(o, wp.POSITION, warm_chunks=warm, compact_window=compact)
        assert W == (C if c < warm else compact)
        _, K, V = chunk(rng, 8, 1, 4)
        o.kv_append(K, V, W)
        ids = sorted(x for x in o.slot_map()[0] if x >= 0)
        assert ids == list(range(max(0, c - W + 1), c + 1)) or (c >= warm and len(ids) <= compact)
    assert sorted(x for x in o.slot_map()[0] if x >= 0) == [12, 13]


def test_memory_policy_is_floor_of_budget_over_slot_bytes():
    """slot = K + V = 2 * H * BPC * B * d * 2 bytes: BASELINE.json configs[1] -> 2*12*192*128*128*2 = 150 994 944 B."""
    o = UFOracle(12, 128, 128, 24480, 3)
    assert wp.slot_bytes(o) == 150_994_944
    assert wp.next_window(o, wp.MEMORY, budget_bytes=150_994_943) == 1           # clamped up to 1
    assert wp.next_window(o, wp.MEMORY, budget_bytes=2 * 150_994_944) == 2
    assert wp.next_window(o, wp.MEMORY, budget_bytes=2 * 150_994_944 - 1) == 1
    assert wp.next_window(o, wp.MEMORY, budget_bytes=10 ** 12) == 3              # clamped to C


def test_usage_statistic_bruteforce_and_content_rule():
    """usage[chunk] = number of (head, query block, kept top-k block) triples whose block lies in the chunk, counted
    with plain loops over the id lists; a chunk whose keys are tiny is never chosen -> share 0 -> the window drops it;
    growing again is allowed afterwards; nothing is dropped at or below compact_window resident chunks."""
    rng = np.random.default_rng(1)
    H, d, B, n, C = 2, 8, 4, 16, 4
    o = UFOracle(H, d, B, n, C, sink_blocks=0)
    windows = []
    for c in range(7):
        W = wp.next_window(o, wp.CONTENT, compact_window=2, min_share_permille=200)
        windows.append(W)
        Q, K, V = chunk(rng, n, H, d, kscale=(1e-3 if c == 1 else 1.0))          # chunk 1's keys score ~0
        Q = bf16(np.abs(Q) + 0.5)
        K = bf16(np.abs(K)) if c != 1 else K
        o.kv_append(K, V, W)
        idx, cnt = o.select_blocks(Q, topk_count=2)
        kept, ids = wp.select_usage(o)
        want = {}
        for h in range(H):
            for i in range(cnt.shape[1]):
                for g in idx[h, i, :cnt[h, i]]:
                    want[int(g) // 4] = want.get(int(g) // 4, 0) + 1
        assert ids == [x for x in sorted(o.slot_map()[0]) if 0 <= x < c]
        assert kept == [want.get(x, 0) for x in ids]
        assert sum(kept) == (H * 4 * min(2, 4 * len(ids)) if ids else 0)
    # chunk 0: nothing measured -> 1; chunk 1: one resident -> 2; chunk 2: chunk 0 well used -> 3; chunk 3: the oldest
    # survivor would be chunk 0 (used) -> 4; before chunk 5 the FIFO victim is chunk 0 and the oldest survivor chunk 1,
    # which no row ever selects -> it goes one append earlier than FIFO would evict it: W = 3
    assert windows[:5] == [1, 2, 3, 4, 3]
    assert 1 not in o.slot_map()[0]


def test_content_rule_bruteforce_state_machine():
    """The rule re-done on plain lists for random usage tables (no oracle state): FIFO victim first, then oldest
    survivors below the share threshold, never below compact_window, never the newest chunk."""
    rng = np.random.default_rng(5)

    class Fake:
        pass

    for _ in range(300):
        C = int(rng.integers(1, 7))
        R = int(rng.integers(1, C + 1))
        nxt = int(rng.integers(R, 40))
        f = Fake()
        f.C, f.next_chunk, f.BPC = C, nxt, 4
        f.resident = [{"id": nxt - R + i} for i in range(R)]
        kept = [int(x) for x in rng.integers(0, 50, R - 1)]
        compact, theta = int(rng.integers(1, C + 1)), int(rng.integers(0, 1001))
        # encode the usage table as an index list the oracle's own counter will read back
        ids = [ch["id"] for ch in f.resident[:-1]]
        flat = [cid * 4 for cid, k in zip(ids, kept) for _ in range(k)]
        f.sel = {"idx": np.asarray(flat, dtype=np.int64).reshape(1, 1, -1), "cnt": np.asarray([[len(flat)]])}
        got = wp.next_window(f, wp.CONTENT, compact_window=compact, min_share_permille=theta)
        survivors = list(zip(ids, kept))
        T = min(C, R + 1)
        if R + 1 > C and survivors:
            survivors = survivors[1:]
        total = sum(kept)
        if total > 0:
            while survivors and T > compact and survivors[0][1] * 1000 // total < theta:
                survivors.pop(0)
                T -= 1
        assert got == max(1, min(C, T)), (C, R, kept, compact, theta, got, T)


@pytest.mark.parametrize("kind", ["position", "memory"])
def test_abi_host_only_policies_match_the_oracle(kind):
    """uf_next_window on a host-only ctx (device = -1) against the oracle over a 20-chunk stream, and the slot maps
    that result from feeding the windows back into uf_kv_append."""
    import paper_2606_09150_b200 as uf
    C = 5
    ctx = uf.uf_ctx_create(3, 64, 64, 640, C, 1, 4, -1)
    o = UFOracle(3, 64, 64, 640, C)
    rng = np.random.default_rng(2)
    try:
        for c in range(20):
            if kind == "position":
                kw = dict(warm_chunks=7, compact_window=2)
                W = uf.uf_next_window(ctx, uf.UF_WIN_POSITION, **kw)
                Wo = wp.next_window(o, wp.POSITION, **kw)
            else:
                budget = int(rng.integers(0, 7)) * wp.slot_bytes(o) + int(rng.integers(0, 1000))
                W = uf.uf_next_window(ctx, uf.UF_WIN_MEMORY, budget_bytes=budget)
                Wo = wp.next_window(o, wp.MEMORY, budget_bytes=budget)
            assert W == Wo
            uf.uf_kv_append(ctx, None, None, 640, 192, 64, W, None)
            o.kv_append(np.zeros((640, 3, 64)), np.zeros((640, 3, 64)), W)
            assert uf.uf_get_slot_map(ctx, C) == o.slot_map()
        assert uf.uf_next_window(ctx, uf.UF_WIN_FIXED) == C
        n_res = uf.uf_get_slot_map(ctx, C)[1]                                     # host-only: nothing measured -> grow
        assert uf.uf_next_window(ctx, uf.UF_WIN_CONTENT, compact_window=1, min_share_permille=500) == min(C, n_res + 1) \
            == wp.next_window(o, wp.CONTENT, compact_window=1, min_share_permille=500)
        with pytest.raises(uf.UFError):
            uf.uf_next_window(ctx, 9)
    finally:
        uf.uf_ctx_destroy(ctx)
