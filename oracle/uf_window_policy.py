"""CPU oracle of the SR cache window policy.

*** TEST INFRASTRUCTURE — NOT A PRODUCT PATH *** (same rules as oracle/uf_oracle.py).

The paper names the idea and gives no rule:
  P:136 (iii)  "SR cache length adaptation. ... generation quality relatively insensitive to KV cache length. We
               exploit this by dynamically selecting a compact cache window, trading minimal quality for significant
               memory and compute savings during extended sequence generation."
  P:353        "SR cache window: dynamically selected based on content complexity."
  P:1103-1104  "(iii) SR cache length adaptation: Select compact SR KV window based on chunk position and memory budget"
Reading R-36: three stated policies, one per hint, each a pure integer function that yields the
`window_chunks` of the NEXT append (the eviction mechanism itself is kv_append's, R-17).  The RULES have nothing
in the paper to be checked against ("parity unpinned" for the rules); what is pinned is that this file computes
what its docstrings say (closed forms and brute-force counts in tests/test_window_policy_pins.py).

  position   W = C for chunks 0 .. warm_chunks-1, compact_window afterwards.
  memory     W = floor(budget_bytes / slot_bytes), slot_bytes = 2 (K, V) * H * BPC * B * d * 2 bytes.
  content    statistic: kept top-k blocks of the last selection per listed chunk, summed over heads and query
             blocks; share[j] = 1000 * kept[j] // total.  T = min(C, resident + 1) chunks would be resident after the
             next append under plain FIFO (its victim, if the cache is full, goes anyway).  Then, oldest survivor
             first: while share < min_share_permille and T > compact_window, that chunk is evicted too (T -= 1).
             W = T.  No selection / no candidates yet: W = min(C, resident + 1).  The newest chunk is never a victim.
All results clamped to 1 .. C.
"""
from __future__ import annotations

import numpy as np

FIXED, POSITION, MEMORY, CONTENT = range(4)


def select_usage(orc):
    """(kept per listed chunk, chunk ids), ascending chunk id, for the oracle's last selection.
    UFOracle: listed = resident chunks older than the newest (the candidates' chunks); only TOPK entries count
    (sink and current chunk are kept unconditionally and say nothing about the cache).
    UFPaperOracle: listed = all resident chunks; every kept block counts (the own block included: it is a member of
    the kept set the kernel emits)."""
    if hasattr(orc, "NB"):                                   # paper-mask oracle
        ids = [ch["id"] for ch in orc.resident]
        kept = {c: 0 for c in ids}
        for row in orc.sel["kept"]:
            for lst in row:
                for g in lst:
                    kept[g // orc.NB] += 1
        return [kept[c] for c in ids], ids
    cur = orc.resident[-1]["id"]
    ids = [ch["id"] for ch in orc.resident if ch["id"] < cur]
    idx, cnt = orc.sel["idx"], orc.sel["cnt"]
    kept = {c: 0 for c in ids}
    H, nqb = cnt.shape
    for h in range(H):
        for i in range(nqb):
            for g in idx[h, i, :cnt[h, i]]:
                kept[int(g) // orc.BPC] += 1
    if not ids or idx.shape[2] == 0:
        return [], []
    return [kept[c] for c in ids], ids


def slot_bytes(orc) -> int:
    """bytes of one cache slot: K and V, H heads, BPC blocks of B rows of d bf16"""
    bpc = orc.NB if hasattr(orc, "NB") else orc.BPC
    B = orc.bt * orc.bh * orc.bw if hasattr(orc, "NB") else orc.B
    return 2 * orc.H * bpc * B * orc.d * 2


def next_window(orc, kind: int, warm_chunks: int = 0, compact_window: int = 1, min_share_permille: int = 0,
                budget_bytes: int = 0) -> int:
    C = orc.C
    clamp = lambda w: max(1, min(C, int(w)))  # noqa: E731
    nxt = orc.next_chunk
    if kind == FIXED:
        return C
    if kind == POSITION:
        return C if nxt < warm_chunks else clamp(compact_window)
    if kind == MEMORY:
        return clamp(budget_bytes // slot_bytes(orc))
    if kind == CONTENT:
        R = len(orc.resident)
        T = clamp(R + 1)
        if orc.sel is None:
            return T
        kept, ids = select_usage(orc)
        total = sum(kept)
        if total == 0:
            return T
        j = 1 if R + 1 > C else 0                          # the FIFO victim is not a survivor
        while (j < len(ids) and ids[j] != nxt - 1 and T > compact_window
               and kept[j] * 1000 // total < min_share_permille):
            T -= 1
            j += 1
        return clamp(T)
    raise ValueError(kind)
