"""Pins for the CPU oracle (oracle/uf_oracle.py) against things other than itself:
closed forms, invariants, brute force with exact rationals / pure-Python loops, an
independently written dense chunk-causal attention (scipy softmax on concatenated tensors),
and the counts BASELINE.json configs[0] fixes (tests/golden/).  CPU only.

Each test names the mistake it is meant to catch.
"""
import itertools
import math
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy.special import logsumexp, softmax

import uf_workloads as wl
from oracle import UFOracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def bf16(x):
    """Round to bf16 and widen back: the oracle always sees exact bf16 values."""
    return wl.bf16_bits_to_f32(wl.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))).astype(np.float64)


def rand_chunk(rng, n, H, d, scale=1.0):
    return tuple(bf16(scale * rng.standard_normal((n, H, d))) for _ in range(3))


def run_stream(orc, chunks, **sel):
    """append -> select -> attention for every chunk; returns per-chunk (idx, cnt, O, lse)."""
    out = []
    for (Q, K, V) in chunks:
        orc.kv_append(K, V)
        idx, cnt = orc.select_blocks(Q, **sel)
        O, lse = orc.sparse_attn(Q)
        out.append((idx, cnt, O, lse))
    return out


# --------------------------------------------------------------------------- cache / slot map

def test_slot_map_closed_form_constant_window():
    """slot = c mod C, resident = last C ids (SURVEY §8(c) pins).  Catches: off-by-one in the
    eviction bound (C counting priors only), wrong free-slot choice."""
    rng = np.random.default_rng(1)
    for C in (1, 2, 3, 4):
        orc = UFOracle(1, 4, 4, 8, C)
        for c in range(20):
            _, K, V = rand_chunk(rng, 8, 1, 4)
            slot = orc.kv_append(K, V)
            assert slot == c % C
            slots, n_res, newest = orc.slot_map()
            assert newest == c and n_res == min(c + 1, C)
            assert sorted(x for x in slots if x >= 0) == list(range(max(0, c - C + 1), c + 1))


def test_window_shrink_is_fifo_and_never_resurrects():
    """Shrinking W evicts several chunks oldest-first; growing W afterwards brings nothing back
    (S8c-17).  Catches: evicting newest, evicting only one, resurrecting."""
    rng = np.random.default_rng(2)
    orc = UFOracle(1, 4, 4, 8, 4)
    for c in range(4):
        orc.kv_append(*rand_chunk(rng, 8, 1, 4)[1:])
    assert orc.slot_map()[0] == [0, 1, 2, 3]
    orc.kv_append(*rand_chunk(rng, 8, 1, 4)[1:], window_chunks=2)        # c = 4: keep {3, 4}
    slots, n_res, newest = orc.slot_map()
    assert n_res == 2 and newest == 4
    assert slots == [4, -1, -1, 3]                                       # lowest free slot reused
    orc.kv_append(*rand_chunk(rng, 8, 1, 4)[1:], window_chunks=4)        # c = 5: W grows
    slots, n_res, _ = orc.slot_map()
    assert slots == [4, 5, -1, 3] and n_res == 3                         # 1, 2 stay gone


def test_slot_invariants_random_windows():
    """Invariants under random windows: a resident chunk never changes slot, no slot is shared,
    resident ids are a contiguous range ending at c of length <= W."""
    rng = np.random.default_rng(3)
    C = 5
    orc = UFOracle(1, 4, 4, 8, C)
    where = {}
    for c in range(60):
        W = int(rng.integers(1, C + 1))
        orc.kv_append(*rand_chunk(rng, 8, 1, 4)[1:], window_chunks=W)
        slots, n_res, newest = orc.slot_map()
        ids = sorted(x for x in slots if x >= 0)
        assert len(ids) == n_res <= W and ids == list(range(c - n_res + 1, c + 1))
        assert min(ids) >= c - W + 1
        for s, cid in enumerate(slots):
            if cid >= 0:
                assert where.setdefault(cid, s) == s
        gone = set(where) - set(ids)
        assert all(g < min(ids) for g in gone)


def test_sink_is_chunk0_block0_forever():
    """Sink = first S*B rows of chunk 0, unchanged after chunk 0 is evicted (S8c-14)."""
    rng = np.random.default_rng(4)
    orc = UFOracle(2, 8, 4, 12, 2, sink_blocks=1)
    first = None
    for c in range(7):
        Q, K, V = rand_chunk(rng, 12, 2, 8)
        if c == 0:
            first = (K[:4].copy(), V[:4].copy())
        orc.kv_append(K, V)
        assert np.array_equal(orc.sink_K, first[0]) and np.array_equal(orc.sink_V, first[1])
    assert 0 not in orc.slot_map()[0]
    kr, vr = orc.block_kv(0, from_sink=True)
    assert np.array_equal(kr, first[0]) and np.array_equal(vr, first[1])


# --------------------------------------------------------------------------- pooling / scores

def test_pooling_constant_and_ragged():
    """Mean of a constant block is the constant, also for the ragged last block (divide by the
    number of valid rows r, not by B — S8c-3).  Catches: dividing by B, pooling over pad rows."""
    orc = UFOracle(2, 4, 8, 24, 2)
    n = 19                                                # blocks of 8, 8, 3
    X = np.zeros((n, 2, 4))
    X[0:8], X[8:16], X[16:19] = 1.5, -2.0, 7.0
    m = orc.pooled_mean(X)
    assert m.shape == (2, 3, 4)
    assert np.all(m[:, 0] == 1.5) and np.all(m[:, 1] == -2.0) and np.all(m[:, 2] == 7.0)


def test_pooling_and_scores_vs_exact_rationals():
    """Pooled means and Eq. 4 scores against exact rational arithmetic on the bf16 inputs.
    Catches: wrong axis, missing 1/sqrt(d), transposed operands."""
    rng = np.random.default_rng(5)
    H, d, B, n = 2, 8, 4, 10
    orc = UFOracle(H, d, B, n, 3)
    Q0, K0, V0 = rand_chunk(rng, n, H, d)
    Q1, K1, V1 = rand_chunk(rng, n, H, d)
    orc.kv_append(K0, V0)
    orc.kv_append(K1, V1)
    qbar = orc.pooled_mean(Q1)
    kbar = orc.pooled_mean(K0)
    for h in range(H):
        for i in range(3):
            rows_q = range(i * B, min((i + 1) * B, n))
            for j in range(3):
                rows_k = range(j * B, min((j + 1) * B, n))
                dot = Fraction(0)
                for t in range(d):
                    qm = sum(Fraction(float(Q1[r, h, t])) for r in rows_q) / len(rows_q)
                    km = sum(Fraction(float(K0[r, h, t])) for r in rows_k) / len(rows_k)
                    assert abs(float(qm) - qbar[h, i, t]) <= 1e-15 * max(1.0, abs(float(qm)))
                    dot += qm * km
                want = float(dot) / math.sqrt(d)
                got = orc.block_scores(qbar[h], kbar[h])[i, j]
                assert abs(got - want) <= 1e-13 * max(1.0, abs(want))


def brute_topk(scores, ids, k):
    """Full sort in pure Python: larger score first, equal scores -> smaller id first."""
    order = sorted(range(len(ids)), key=lambda j: (-scores[j], ids[j]))
    return sorted(ids[j] for j in order[:k])


def test_topk_vs_bruteforce_full_sort_exact():
    """Selection against a pure-Python full sort over exact rational scores.
    Catches: ascending-vs-descending, tie rule, candidate set (sink / current excluded)."""
    rng = np.random.default_rng(6)
    H, d, B, n, C = 2, 8, 4, 12, 4
    orc = UFOracle(H, d, B, n, C)
    chunks = [rand_chunk(rng, n, H, d) for _ in range(4)]
    for c, (Q, K, V) in enumerate(chunks):
        orc.kv_append(K, V)
        idx, cnt = orc.select_blocks(Q, topk_count=3)
        cand = orc.candidate_ids()
        bpc = 3
        want_cand = [g for g in range(c * bpc) if g >= 1]              # all prior blocks minus sink id 0
        assert cand == want_cand
        for h in range(H):
            for i in range(bpc):
                sc = []
                for g in cand:
                    cg, b = divmod(g, bpc)
                    Kg = chunks[cg][1]
                    dot = Fraction(0)
                    for t in range(d):
                        qm = sum(Fraction(float(x)) for x in Q[i * B:(i + 1) * B, h, t]) / B
                        km = sum(Fraction(float(x)) for x in Kg[b * B:(b + 1) * B, h, t]) / B
                        dot += qm * km
                    sc.append(dot)
                k = min(3, len(cand))
                assert cnt[h, i] == k
                assert list(idx[h, i, :k]) == brute_topk(sc, cand, k)


def test_topk_invariants_and_threshold_property():
    """TOPK subset of CAND, |TOPK| = min(k,|CAND|), ascending ids, and every kept score >= every
    dropped score."""
    rng = np.random.default_rng(7)
    H, d, B, n, C = 3, 16, 8, 40, 4
    orc = UFOracle(H, d, B, n, C, k_min=2)
    for c in range(5):
        Q, K, V = rand_chunk(rng, n, H, d)
        orc.kv_append(K, V)
        idx, cnt = orc.select_blocks(Q, topk_percent=30)
        cand = orc.candidate_ids()
        k = min(max(2, (30 * len(cand)) // 100), len(cand))
        assert np.all(cnt == k)
        if not cand:
            continue
        qbar = orc.pooled_mean(Q)
        kbar = np.stack([np.stack([orc.block_kv(g)[0][:, h].mean(0) for g in cand]) for h in range(H)])
        for h in range(H):
            s = qbar[h] @ kbar[h].T
            for i in range(idx.shape[1]):
                kept = list(idx[h, i, :k])
                assert kept == sorted(set(kept)) and set(kept) <= set(cand)
                pos = [cand.index(g) for g in kept]
                drop = [j for j in range(len(cand)) if j not in pos]
                if drop and pos:
                    assert s[i, pos].min() >= s[i, drop].max() - 1e-12


def test_duplicate_blocks_tie_goes_to_lower_id():
    """Bitwise-duplicated key blocks score equal; with room for one, the lower id is kept (BJ)."""
    rng = np.random.default_rng(8)
    H, d, B, n = 1, 8, 4, 16                                            # 4 blocks / chunk
    orc = UFOracle(H, d, B, n, 3)
    Q0, K0, V0 = rand_chunk(rng, n, H, d)
    blk = bf16(3.0 + rng.standard_normal((B, H, d)))                    # a strong block
    K0[4:8] = blk                                                       # g = 1
    K0[12:16] = blk                                                     # g = 3 (copy)
    orc.kv_append(K0, V0)
    Q1, K1, V1 = rand_chunk(rng, n, H, d)
    Q1[:] = bf16(np.abs(Q1))                                            # positive q -> blk scores highest
    orc.kv_append(K1, V1)
    idx, cnt = orc.select_blocks(Q1, topk_count=1)
    assert np.all(cnt == 1) and np.all(idx[..., 0] == 1)
    idx2, _ = orc.select_blocks(Q1, topk_count=2)
    assert np.all(idx2[..., 0] == 1) and np.all(idx2[..., 1] == 3)


def test_selection_invariant_to_positive_q_scale_and_k_saturation():
    """Scaling Q by 2 (exact in binary fp) keeps every selection; k >= |CAND| keeps all."""
    rng = np.random.default_rng(9)
    H, d, B, n = 2, 16, 8, 48
    orc = UFOracle(H, d, B, n, 3)
    for c in range(3):
        Q, K, V = rand_chunk(rng, n, H, d)
        orc.kv_append(K, V)
    a, _ = orc.select_blocks(Q, topk_count=4)
    b, _ = orc.select_blocks(2.0 * Q, topk_count=4)
    assert np.array_equal(a, b)
    allc, cnt = orc.select_blocks(Q, topk_count=10 ** 6)
    cand = orc.candidate_ids()
    assert np.all(cnt == len(cand)) and np.all(allc == np.asarray(cand)[None, None, :])


def test_percent_budget_integer_floor_and_kmin():
    """k = max(k_min, floor(pct*|CAND|/100)) clamped to |CAND| (S8c-9): the BJ configs give
    48 / 101 / 96 / 76."""
    orc = UFOracle(1, 4, 4, 8, 2, k_min=4)
    assert orc.topk_budget(192, topk_percent=25) == 48
    assert orc.topk_budget(676, topk_percent=15) == 101
    assert orc.topk_budget(384, topk_percent=25) == 96
    assert orc.topk_budget(384, topk_percent=20) == 76
    assert orc.topk_budget(10, topk_percent=25) == 4          # k_min floor
    assert orc.topk_budget(3, topk_percent=25) == 3           # clamp to |CAND|
    assert orc.topk_budget(0, topk_percent=25) == 0
    assert orc.topk_budget(3, topk_count=2) == 2 and orc.topk_budget(1, topk_count=2) == 1


def test_golden_config0_counts():
    """BASELINE.json configs[0]: kept-block counts 2, 4, 5 and candidate sets per chunk."""
    w = wl.CONFIGS["tiny"]
    rows = [l.split() for l in open(os.path.join(GOLDEN, "config0_kept_blocks.txt")) if l[0] != "#"]
    orc = UFOracle(w.n_heads, w.head_dim, w.block, w.chunk_tokens, w.capacity_chunks, w.sink_blocks)
    for (c, n_cand, k_eff, kept, cands), (Qb, Kb, Vb) in zip(rows, wl.make_stream(w, 3)):
        Q, K, V = (wl.bf16_bits_to_f32(x) for x in (Qb, Kb, Vb))
        orc.kv_append(K, V)
        idx, cnt = orc.select_blocks(Q, topk_count=w.topk_count)
        want_c = [] if cands == "-" else [int(x) for x in cands.split(",")]
        assert orc.candidate_ids() == want_c and len(want_c) == int(n_cand)
        assert np.all(cnt == int(k_eff))
        for i in range(w.bpc):
            ids = [g for g, _ in orc.kept_blocks(0, i)]
            assert len(ids) == int(kept) == len(set(ids))
            assert set(orc.current_ids()) <= set(ids)
            if int(c) > 0:
                assert 0 in ids
    assert list(idx[0, 0]) != [] and set(idx[0, 0]) <= {1, 2, 3}


# --------------------------------------------------------------------------- attention

def dense_chunk_causal(chunks, c, scale=None):
    """Independent reference: chunk c's queries attend to ALL tokens of chunks 0..c (bidirectional
    inside chunk c, nothing later) — scipy softmax over concatenated tensors, no blocks."""
    Q = chunks[c][0]
    K = np.concatenate([ch[1] for ch in chunks[:c + 1]], axis=0)
    V = np.concatenate([ch[2] for ch in chunks[:c + 1]], axis=0)
    d = Q.shape[-1]
    sc = (1.0 / math.sqrt(d)) if scale is None else scale
    logits = np.einsum("nhd,mhd->hnm", Q, K) * sc
    P = softmax(logits, axis=-1)
    return np.einsum("hnm,mhd->nhd", P, V), logsumexp(logits, axis=-1)


@pytest.mark.parametrize("n", [24, 21])                                  # whole blocks / ragged tail
def test_all_kept_equals_dense_chunk_causal(n):
    """BJ pin: an all-kept mask must equal dense causal attention.  With capacity >= stream length
    and k >= |CAND| every earlier block is kept (sink + topk + current cover all).  Catches:
    dropped blocks, double-counted sink, ragged rows, wrong scale, softmax axis."""
    rng = np.random.default_rng(10)
    H, d, B = 2, 16, 8
    chunks = [rand_chunk(rng, n, H, d) for _ in range(4)]
    orc = UFOracle(H, d, B, n, capacity_chunks=4)
    res = run_stream(orc, chunks, topk_count=10 ** 6)
    for c in range(4):
        want, want_lse = dense_chunk_causal(chunks, c)
        assert np.allclose(res[c][2], want, rtol=0, atol=1e-12)
        assert np.allclose(res[c][3], want_lse, rtol=0, atol=1e-12)


def test_custom_softmax_scale():
    rng = np.random.default_rng(11)
    chunks = [rand_chunk(rng, 16, 1, 8) for _ in range(2)]
    orc = UFOracle(1, 8, 8, 16, 2)
    for c, (Q, K, V) in enumerate(chunks):
        orc.kv_append(K, V)
        orc.select_blocks(Q, topk_count=99)
        O, _ = orc.sparse_attn(Q, softmax_scale=0.3)
        assert np.allclose(O, dense_chunk_causal(chunks, c, scale=0.3)[0], atol=1e-12)


def test_rows_sum_to_one_and_constant_v():
    """V == const -> O == const (softmax rows sum to 1)."""
    rng = np.random.default_rng(12)
    H, d, B, n = 2, 8, 4, 14
    orc = UFOracle(H, d, B, n, 2)
    for c in range(4):
        Q, K, V = rand_chunk(rng, n, H, d, scale=3.0)
        V[:] = 0.75
        orc.kv_append(K, V)
        orc.select_blocks(Q, topk_count=1)
        O, _ = orc.sparse_attn(Q)
        assert np.allclose(O, 0.75, rtol=0, atol=1e-14)


def test_zero_q_gives_mean_of_kept_values():
    """Q == 0 -> uniform softmax -> O = mean of V over the kept VALID keys (closed form).
    Catches: pad rows counted as keys, sink counted twice."""
    rng = np.random.default_rng(13)
    H, d, B, n = 1, 8, 4, 10                                            # ragged: 4, 4, 2
    orc = UFOracle(H, d, B, n, 2)
    chunks = [rand_chunk(rng, n, H, d) for _ in range(3)]
    for c, (Q, K, V) in enumerate(chunks):
        orc.kv_append(K, V)
        orc.select_blocks(0 * Q, topk_count=1)
        O, _ = orc.sparse_attn(0 * Q)
        for i in range(3):
            rows = []
            for g, fs in orc.kept_blocks(0, i):
                cg, b = divmod(g, 3)
                rows.append(chunks[cg][2][b * B:min((b + 1) * B, n), 0])
            want = np.concatenate(rows).mean(axis=0)
            assert np.allclose(O[i * B:min((i + 1) * B, n), 0], want, atol=1e-14)


def test_indicator_v_mass_only_on_kept_blocks_and_never_future():
    """V channel j = 1 on tokens of global block j: O[:, j] is the attention mass on block j.
    It must be exactly 0 on every non-kept block, sum to 1 over kept ones, and no kept id may
    belong to a later chunk (block-causality)."""
    rng = np.random.default_rng(14)
    H, B, n, C = 2, 4, 12, 3                                            # BPC = 3
    n_chunks = 4
    d = 3 * n_chunks                                                    # one channel per global block
    orc = UFOracle(H, d, B, n, C)
    for c in range(n_chunks):
        Q, K, _ = rand_chunk(rng, n, H, d, scale=2.0)
        V = np.zeros((n, H, d))
        for b in range(3):
            V[b * B:(b + 1) * B, :, c * 3 + b] = 1.0
        orc.kv_append(K, V)
        idx, cnt = orc.select_blocks(Q, topk_count=2)
        O, _ = orc.sparse_attn(Q)
        for h in range(H):
            for i in range(3):
                kept = {g for g, _ in orc.kept_blocks(h, i)}
                assert max(kept) < (c + 1) * 3
                o = O[i * B:(i + 1) * B, h]
                assert np.allclose(o.sum(axis=1), 1.0, atol=1e-14)
                for g in range(d):
                    if g not in kept:
                        assert np.all(o[:, g] == 0.0)
                    else:
                        assert np.all(o[:, g] > 0.0)


def test_key_shift_invariance():
    """Adding one constant vector u to every key changes q.k by q.u for all keys of a row:
    softmax, hence O, is unchanged; block scores shift by qbar.u per row, so the selection is
    unchanged too.  Catches: per-block (instead of per-row) max, missing terms."""
    rng = np.random.default_rng(15)
    H, d, B, n = 2, 8, 4, 12
    u = np.array([0.5, -1.0, 0.25, 2.0, -0.5, 1.0, 0.0, -2.0])          # exact in bf16
    chunks = [rand_chunk(rng, n, H, d) for _ in range(3)]
    a = UFOracle(H, d, B, n, 3)
    b = UFOracle(H, d, B, n, 3)
    for (Q, K, V) in chunks:
        a.kv_append(K, V)
        b.kv_append(K + u, V)
        ia, _ = a.select_blocks(Q, topk_count=2)
        ib, _ = b.select_blocks(Q, topk_count=2)
        assert np.array_equal(ia, ib)
        assert np.allclose(a.sparse_attn(Q)[0], b.sparse_attn(Q)[0], atol=1e-11)


def test_kept_order_permutation_invariance():
    rng = np.random.default_rng(16)
    H, d, B, n = 1, 8, 4, 12
    orc = UFOracle(H, d, B, n, 3)
    for c in range(3):
        Q, K, V = rand_chunk(rng, n, H, d)
        orc.kv_append(K, V)
    orc.select_blocks(Q, topk_count=3)
    O1, _ = orc.sparse_attn(Q)
    orig = orc.kept_blocks
    orc.kept_blocks = lambda h, i: list(reversed(orig(h, i)))
    O2, _ = orc.sparse_attn(Q)
    assert np.allclose(O1, O2, atol=1e-13)


def test_attention_vs_pure_python_bruteforce():
    """Whole path on a tiny case re-done with Python loops and math.exp from the definitions."""
    rng = np.random.default_rng(17)
    H, d, B, n, C, k = 1, 4, 2, 5, 2, 1                                 # BPC = 3, ragged (2,2,1)
    chunks = [rand_chunk(rng, n, H, d) for _ in range(4)]
    orc = UFOracle(H, d, B, n, C)
    res = run_stream(orc, chunks, topk_count=k)
    bpc = 3
    for c in range(4):
        Q = chunks[c][0]
        resident = [x for x in (c - 1,) if x >= 0]                       # C = 2 -> one prior chunk
        sink = [0] if c > 0 else []
        cand = [cc * bpc + b for cc in resident for b in range(bpc) if cc * bpc + b not in (0,)]

        def rows_of(g):
            cg, b = divmod(g, bpc)
            return cg, range(b * B, min((b + 1) * B, n))

        for i in range(bpc):
            qrows = range(i * B, min((i + 1) * B, n))
            qm = [sum(Q[r, 0, t] for r in qrows) / len(qrows) for t in range(d)]
            sc = []
            for g in cand:
                cg, rr = rows_of(g)
                km = [sum(chunks[cg][1][r, 0, t] for r in rr) / len(rr) for t in range(d)]
                sc.append(sum(qm[t] * km[t] for t in range(d)) / math.sqrt(d))
            top = brute_topk(sc, cand, min(k, len(cand)))
            assert list(res[c][0][0, i, :len(top)]) == top
            kept = sink + top + [c * bpc + b for b in range(bpc)]
            for r in qrows:
                logit, vals = [], []
                for g in kept:
                    cg, rr = rows_of(g)
                    for m in rr:
                        logit.append(sum(Q[r, 0, t] * chunks[cg][1][m, 0, t] for t in range(d)) / math.sqrt(d))
                        vals.append(chunks[cg][2][m, 0])
                mx = max(logit)
                e = [math.exp(x - mx) for x in logit]
                z = sum(e)
                want = sum(ei * v for ei, v in zip(e, vals)) / z
                assert np.allclose(res[c][2][r, 0], want, atol=1e-13)
                assert abs(res[c][3][0, r] - (mx + math.log(z))) < 1e-13


@pytest.mark.parametrize("S,n0,C", [(0, 5, 2), (0, 5, 3), (2, 5, 2), (2, 5, 3), (2, 3, 2), (3, 3, 3), (1, 1, 2)])
def test_sink_variants_vs_pure_python_bruteforce(S, n0, C):
    """S = 0 (no sink), S >= 2, and a chunk 0 shorter than S*B (the sink is then all of chunk 0, its last
    block ragged): SINK / CAND / KEPT sets, the selection and the attention re-done from the definitions with
    Python loops (readings R-14/R-15: sink = blocks 0..S-1 of chunk 0 that exist, always attended for c > 0,
    never a candidate, never counted twice; served from the sink copy after chunk 0 is evicted).  Catches: a sink
    id left in CAND, a sink block attended twice while chunk 0 is resident, pad rows of a short sink block
    counted as keys, sink dropped after eviction, S = 0 still reserving block 0."""
    rng = np.random.default_rng(100 + 10 * S + n0 + C)
    H, d, B, n, k = 1, 4, 2, 5, 2                                        # BPC = 3, ragged (2, 2, 1)
    bpc = 3
    lens = [n0, n, n, 4, n]
    chunks = [rand_chunk(rng, m, H, d) for m in lens]
    orc = UFOracle(H, d, B, n, C, sink_blocks=S)
    res = run_stream(orc, chunks, topk_count=k)
    sink_tok = min(S * B, n0)
    sink_ids = list(range(-(-sink_tok // B)))                            # blocks of chunk 0 inside the sink

    def rows_of(g):
        cg, b = divmod(g, bpc)
        return cg, range(b * B, min((b + 1) * B, lens[cg]))

    for c in range(len(lens)):
        Q = chunks[c][0]
        resident_prior = [x for x in range(max(0, c - C + 1), c)]
        sink = sink_ids if c > 0 else []
        cand = [cc * bpc + b for cc in resident_prior for b in range(-(-lens[cc] // B))
                if cc * bpc + b not in sink_ids]
        assert orc_sets_equal(res[c], cand, k)
        nqb = -(-lens[c] // B)
        for i in range(nqb):
            qrows = range(i * B, min((i + 1) * B, lens[c]))
            qm = [sum(Q[r, 0, t] for r in qrows) / len(qrows) for t in range(d)]
            sc = []
            for g in cand:
                cg, rr = rows_of(g)
                km = [sum(chunks[cg][1][r, 0, t] for r in rr) / len(rr) for t in range(d)]
                sc.append(sum(qm[t] * km[t] for t in range(d)) / math.sqrt(d))
            top = brute_topk(sc, cand, min(k, len(cand)))
            assert list(res[c][0][0, i, :len(top)]) == top
            # keys: sink rows (from chunk 0's first sink_tok rows), top-k blocks, the whole current chunk
            keys = []
            for g in sink:
                keys += [(0, m) for m in range(g * B, min((g + 1) * B, sink_tok))]
            for g in top:
                cg, rr = rows_of(g)
                keys += [(cg, m) for m in rr]
            keys += [(c, m) for m in range(lens[c])]
            assert len(keys) == len(set(keys)), "a key row is attended twice"
            for r in qrows:
                logit = [sum(Q[r, 0, t] * chunks[cg][1][m, 0, t] for t in range(d)) / math.sqrt(d) for cg, m in keys]
                mx = max(logit)
                e = [math.exp(x - mx) for x in logit]
                z = sum(e)
                want = sum(ei * chunks[cg][2][m, 0] for ei, (cg, m) in zip(e, keys)) / z
                assert np.allclose(res[c][2][r, 0], want, atol=1e-13)
                assert abs(res[c][3][0, r] - (mx + math.log(z))) < 1e-13


def orc_sets_equal(step_result, cand, k):
    """count column of a step == min(k, |CAND|) for every (head, query block)"""
    return bool(np.all(step_result[1] == min(k, len(cand))))


def test_sink_candidate_and_kept_sets_explicit():
    """The sets themselves, spelled out for S = 0 / 2 and a short chunk 0 (B = 4, BPC = 3, C = 2)."""
    rng = np.random.default_rng(77)
    H, d, B, n = 1, 4, 4, 12
    # S = 0: nothing reserved, block 0 of chunk 0 is an ordinary candidate while chunk 0 is resident
    o = UFOracle(H, d, B, n, 2, sink_blocks=0)
    for c in range(3):
        Q, K, V = rand_chunk(rng, n, H, d)
        o.kv_append(K, V)
        o.select_blocks(Q, topk_count=1)
        assert o.sink_ids() == []
        assert o.candidate_ids() == ([] if c == 0 else list(range((c - 1) * 3, c * 3)))
        assert [g for g, fs in o.kept_blocks(0, 0) if fs] == []
        assert len(o.kept_blocks(0, 0)) == (3 if c == 0 else 4)
    # S = 2: ids 0, 1 are sink; chunk 1 sees CAND = {2} only; after eviction of chunk 0 the sink stays
    o = UFOracle(H, d, B, n, 2, sink_blocks=2)
    for c in range(3):
        Q, K, V = rand_chunk(rng, n, H, d)
        o.kv_append(K, V)
        o.select_blocks(Q, topk_count=5)
        assert o.sink_ids() == [0, 1]
        assert o.candidate_ids() == [[], [2], [3, 4, 5]][c]
        kept = o.kept_blocks(0, 1)
        assert [g for g, fs in kept if fs] == ([] if c == 0 else [0, 1])
        assert [g for g, fs in kept if not fs] == [[0, 1, 2], [2, 3, 4, 5], [3, 4, 5, 6, 7, 8]][c]
    # chunk 0 of 6 tokens with S = 2: the sink is rows 0..5 (block 1 ragged, 2 rows); no candidate from chunk 0
    o = UFOracle(H, d, B, n, 2, sink_blocks=2)
    Q, K, V = rand_chunk(rng, 6, H, d)
    o.kv_append(K, V)
    assert o.sink_K.shape[0] == 6 and o.sink_ids() == [0, 1]
    Q, K, V = rand_chunk(rng, n, H, d)
    o.kv_append(K, V)
    o.select_blocks(Q, topk_count=3)
    assert o.candidate_ids() == [] and o.sel["cnt"].max() == 0
    kr, vr = o.block_kv(1, from_sink=True)
    assert kr.shape[0] == 2
    assert sum(o.block_kv(g, fs)[0].shape[0] for g, fs in o.kept_blocks(0, 0)) == 6 + n


def test_kept_flop_closed_form():
    """kept_flop = 4 d sum(rows x keys): all blocks full -> 4 d H n (S B + k B + n)."""
    rng = np.random.default_rng(78)
    H, d, B, n = 2, 4, 4, 12
    o = UFOracle(H, d, B, n, 3, sink_blocks=1)
    for c in range(3):
        Q, K, V = rand_chunk(rng, n, H, d)
        o.kv_append(K, V)
    o.select_blocks(Q, topk_count=2)
    assert o.kept_flop() == 4 * d * H * n * (1 * B + 2 * B + n)


def test_sparse_differs_from_dense_when_blocks_dropped():
    """Sanity: with k small the result is NOT the dense one (the mask really restricts)."""
    rng = np.random.default_rng(18)
    chunks = [rand_chunk(rng, 32, 1, 8) for _ in range(3)]
    orc = UFOracle(1, 8, 4, 32, 3)
    res = run_stream(orc, chunks, topk_count=1)
    assert np.abs(res[2][2] - dense_chunk_causal(chunks, 2)[0]).max() > 1e-3


# --------------------------------------------------------------------------- workload generator

def test_paper_shape_facts():
    for line in open(os.path.join(GOLDEN, "paper_shape_facts.txt")):
        if line.startswith("#"):
            continue
        hp, wp, gh, gw, per = (int(x) for x in line.split())
        assert wl.token_grid(hp, wp) == (gh, gw) and gh * gw == per
    assert wl.CONFIGS["1k"].chunk_tokens == 24480 and wl.CONFIGS["1k"].bpc == 192
    assert wl.CONFIGS["2k"].chunk_tokens == 43200 and wl.CONFIGS["2k"].bpc == 338
    assert -(-2 * 6240 // 128) == 98                                    # P:820 "N_blocks ~ 200" = 2 x 98


def test_bf16_rounding_is_rne_and_roundtrips():
    x = np.array([1.0, 1.00390625, 1.01171875, -2.5, 3.1415927, 1e-8, 65504.0], dtype=np.float32)
    b = wl.f32_to_bf16_bits(x)
    y = wl.bf16_bits_to_f32(b)
    assert y[0] == 1.0 and y[3] == -2.5
    assert y[1] == 1.0                      # 1 + 2^-8 is a tie -> even mantissa (1.0)
    assert y[2] == np.float32(1.015625)     # 1 + 3*2^-8 is a tie -> even mantissa (1 + 2^-6)
    assert np.all(np.abs(y - x) <= np.abs(x) * 2.0 ** -8)
    assert np.array_equal(wl.f32_to_bf16_bits(y), b)


def test_generator_is_seeded_and_shaped():
    w = wl.scaled(wl.CONFIGS["1k"], "1k_small", grid_h=4, grid_w=6, n_heads=2)
    a = wl.make_chunk(w, 1)
    b = wl.make_chunk(w, 1)
    c = wl.make_chunk(w, 2)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    assert not np.array_equal(a[0], c[0])
    assert a[0].shape == (72, 2, 128) and a[0].dtype == np.uint16
    q = wl.bf16_bits_to_f32(a[0]).astype(np.float64)
    assert 1.5 < q.std() < 2.2              # N(0,1) + 2*sin(.) -> variance 1 + 2 = 3
