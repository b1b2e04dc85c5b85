"""CPU oracle for Ultra Flash's sparse causal chunk attention (arxiv/paper_2606_09150).

*** TEST INFRASTRUCTURE — NOT A PRODUCT PATH. ***
Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import this package.  It shares no code with `paper_2606_09150_b200/` (the CUDA path)
and imports nothing from it.  It is deliberately plain and slow: NumPy, fp64 throughout,
no blocking / fusion / online softmax — each function follows the cited passage step by step
so it can be checked against the paper by eye.

Citations: `P:NNN` = line NNN of /root/reference/PAPER.md; `BJ` = BASELINE.json (`north_star`,
`configs`); `S8c-n` = reading n of SURVEY.md §8(c), restated in DESIGN.md §"Readings".

What the path computes, per streaming chunk c (P:86-90, P:136 (iii)):
  1. kv_append   — put the chunk's K,V into a bounded rolling cache, evict under a FIFO window,
                   keep a permanent sink (BJ: "uf_kv_append ... evict under the paper's dynamic
                   cache policy"; P:136 (iii) "dynamically selecting a compact cache window";
                   P:343 "KV cache: 3 temporal windows").
  2. select      — "we pool Q and K within each block, compute block-level attention scores,
                   and retain the top-k most relevant blocks per head", Eq. 4:
                   s_ij^h = qbar_i^h . kbar_j^h / sqrt(d_h), block-mean pooled.
  3. sparse attn — softmax(q k^T / sqrt(d)) v restricted to the kept key blocks, chunk-
                   causal: "each temporal chunk attends only to current and preceding chunks"
                   (P:86); bidirectional inside the current chunk (S8c-18).

Pin status (tests/test_oracle_pins.py, all `-m "not gpu"`):
  kv_append / slot map      pinned: closed form slot = c mod C, resident = last C ids, FIFO shrink,
                            sink bytes constant, brute-force state machine.
  pooled means              pinned: constant block, ragged block divides by r, brute force.
  block scores / top-k      pinned: brute-force full sort, invariants (subset, size, threshold),
                            duplicated blocks -> lower id, positive scaling of Q, k >= |CAND|,
                            BJ config-0 golden counts (tests/golden/config0_kept_blocks.txt).
  sparse attention          pinned: all-kept == independent dense chunk-causal attention
                            (scipy.special.softmax + einsum on concatenated tensors), rows sum to 1,
                            V = const, Q = 0 -> mean of V, indicator-V block mass (causality and
                            sparsity), key-shift invariance, kept-order permutation, brute force.
  Eq. 10 adaptive budget    NOT IMPLEMENTED here (formula inconsistent, S8c-8): parity unpinned
                            for that row; k comes from BJ (count or percent of |CAND|).
"""
from __future__ import annotations

import math

import numpy as np


class UFOracle:
    """State = resident chunks (ascending id) + sink copy.  All tensors fp64, shape [n, H, d].

    Notation: H heads, d head_dim, B block, BPC = ceil(chunk_tokens_max / B),
    C capacity in chunks counting the just-appended one (S8c-16), S sink blocks,
    global key-block id g = chunk * BPC + b.
    """

    def __init__(self, n_heads: int, head_dim: int, block: int, chunk_tokens_max: int,
                 capacity_chunks: int, sink_blocks: int = 1, k_min: int = 4):
        self.H, self.d, self.B = n_heads, head_dim, block
        self.N_max = chunk_tokens_max
        self.BPC = -(-chunk_tokens_max // block)
        self.C, self.S, self.k_min = capacity_chunks, sink_blocks, k_min
        self.reset()

    # ------------------------------------------------------------------ state
    def reset(self) -> None:
        """Start a new video stream: empty cache, no sink (S8c-27)."""
        self.resident: list[dict] = []            # ascending chunk id
        self.slot_chunk = [-1] * self.C           # slot -> chunk id or -1
        self.next_chunk = 0
        self.sink_K = None                        # fp64 [n_sink_tokens, H, d]
        self.sink_V = None
        self.sel = None                           # last selection (lists of global ids)

    def n_blocks(self, n_tokens: int) -> int:
        return -(-n_tokens // self.B)

    # ----------------------------------------------------------------- step 1
    def kv_append(self, K: np.ndarray, V: np.ndarray, window_chunks: int = 0) -> int:
        """Append chunk c = next id; evict; return the slot it went to.

        P:136 (iii); BJ configs[3] ("eviction of the oldest non-sink chunk
        after each append").  Readings S8c-16/17: C counts the current chunk; with window
        W (0 -> C) every resident chunk with id <= c - W is evicted, oldest first; shrinking W
        evicts several, growing never resurrects.  The chunk takes the lowest-numbered free slot.
        On c = 0 its first S blocks are copied to the sink region (S8c-14: sink = chunk 0,
        blocks 0..S-1, kept forever)."""
        K = np.asarray(K, dtype=np.float64)
        V = np.asarray(V, dtype=np.float64)
        n = K.shape[0]
        assert K.shape == V.shape == (n, self.H, self.d) and 1 <= n <= self.N_max
        c = self.next_chunk
        W = self.C if window_chunks in (0, None) else window_chunks
        assert 1 <= W <= self.C
        # evict: ids <= c - W, oldest first
        while self.resident and self.resident[0]["id"] <= c - W:
            gone = self.resident.pop(0)
            self.slot_chunk[gone["slot"]] = -1
        slot = self.slot_chunk.index(-1)          # lowest-numbered free slot
        self.slot_chunk[slot] = c
        self.resident.append({"id": c, "slot": slot, "K": K.copy(), "V": V.copy(), "n": n})
        if c == 0:
            ns = min(self.S * self.B, n)
            self.sink_K, self.sink_V = K[:ns].copy(), V[:ns].copy()
        self.next_chunk = c + 1
        self.sel = None
        return slot

    def slot_map(self):
        """(slot -> chunk id list, number resident, newest chunk id)."""
        return list(self.slot_chunk), len(self.resident), self.next_chunk - 1

    def sink_ids(self) -> list[int]:
        """Global ids of the sink blocks: blocks 0..S-1 of chunk 0 that exist (S8c-14)."""
        if self.sink_K is None:
            return []
        return list(range(self.n_blocks(self.sink_K.shape[0])))

    def candidate_ids(self) -> list[int]:
        """CAND, ascending: blocks of resident chunks older than the current one, minus SINK
        (S8c-10, S8c-15).  No block of a later chunk exists in the state: causality."""
        cur = self.resident[-1]["id"]
        sink = set(self.sink_ids())
        out = []
        for ch in self.resident:
            if ch["id"] < cur:
                for b in range(self.n_blocks(ch["n"])):
                    g = ch["id"] * self.BPC + b
                    if g not in sink:
                        out.append(g)
        return out

    def current_ids(self) -> list[int]:
        ch = self.resident[-1]
        return [ch["id"] * self.BPC + b for b in range(self.n_blocks(ch["n"]))]

    def block_kv(self, g: int, from_sink: bool = False):
        """Valid rows of key block g: (K rows, V rows), fp64 [r, H, d]."""
        if from_sink:
            lo = g * self.B
            return self.sink_K[lo:lo + self.B], self.sink_V[lo:lo + self.B]
        cid, b = divmod(g, self.BPC)
        for ch in self.resident:
            if ch["id"] == cid:
                lo = b * self.B
                return ch["K"][lo:lo + self.B], ch["V"][lo:lo + self.B]
        raise KeyError(f"block {g} (chunk {cid}) is not resident")

    # ----------------------------------------------------------------- step 2
    def pooled_mean(self, X: np.ndarray) -> np.ndarray:
        """Block-mean pooling: mean over the VALID rows of each block (S8c-3).
        X fp64 [n, H, d] -> [H, nblk, d]."""
        n = X.shape[0]
        nb = self.n_blocks(n)
        out = np.empty((self.H, nb, self.d), dtype=np.float64)
        for b in range(nb):
            rows = X[b * self.B:min((b + 1) * self.B, n)]          # [r, H, d]
            out[:, b, :] = rows.sum(axis=0) / float(rows.shape[0])
        return out

    def block_scores(self, qbar: np.ndarray, kbar: np.ndarray) -> np.ndarray:
        """Eq. 4: s_ij = qbar_i . kbar_j / sqrt(d), fp64.  The dot product is the plain
        definition sum_{t=0}^{d-1} qbar_i[t] * kbar_j[t], terms added in index order, each
        multiply and each add rounded once (no fused multiply-add) — stated so that the value,
        hence the top-k decision, is a fixed function of the inputs (S8c-4).
        qbar [nq, d], kbar [nc, d] -> [nq, nc]."""
        s = np.zeros((qbar.shape[0], kbar.shape[0]), dtype=np.float64)
        for t in range(self.d):
            s = s + np.multiply.outer(qbar[:, t], kbar[:, t])
        return s / math.sqrt(float(self.d))

    def topk_budget(self, n_cand: int, topk_count: int = -1, topk_percent: int = -1) -> int:
        """k' = min(k, |CAND|); k = count, or max(k_min, floor(pct * |CAND| / 100)) in integer
        arithmetic (S8c-8/9/10; k_min = 4 from P:818 applies in percent mode only)."""
        if topk_count is not None and topk_count >= 0:
            k = topk_count
        else:
            assert 0 <= topk_percent <= 100
            k = max(self.k_min, (topk_percent * n_cand) // 100)
        return min(k, n_cand)

    def select_blocks(self, Q: np.ndarray, topk_count: int = -1, topk_percent: int = -1):
        """Per head h and query block i keep the k' candidates with the largest score; among equal
        scores the smaller global id wins (BJ; S8c-6/12); emit ascending by id.

        Returns idx int32 [H, nqb, k'] (global ids, ascending) and cnt int32 [H, nqb] (= k')."""
        Q = np.asarray(Q, dtype=np.float64)
        cur = self.resident[-1]
        assert Q.shape == (cur["n"], self.H, self.d)
        cand = self.candidate_ids()
        kk = self.topk_budget(len(cand), topk_count, topk_percent)
        nqb = self.n_blocks(cur["n"])
        idx = np.zeros((self.H, nqb, kk), dtype=np.int32)
        cnt = np.full((self.H, nqb), kk, dtype=np.int32)
        self.min_gap = math.inf                    # diagnostic: smallest k-th/(k+1)-th score gap
        if kk > 0:
            qbar = self.pooled_mean(Q)                                           # [H, nqb, d]
            kbar = np.empty((self.H, len(cand), self.d), dtype=np.float64)
            for j, g in enumerate(cand):
                kr, _ = self.block_kv(g)
                kbar[:, j, :] = kr.sum(axis=0) / float(kr.shape[0])
            cand_arr = np.asarray(cand, dtype=np.int64)
            for h in range(self.H):
                s = self.block_scores(qbar[h], kbar[h]) + 0.0                    # [nqb, |CAND|]
                # stable sort of -s over candidates already in ascending id: ties -> lower id
                order = np.argsort(-s, axis=1, kind="stable")
                top = np.sort(order[:, :kk], axis=1)
                idx[h] = cand_arr[top].astype(np.int32)
                if kk < len(cand):
                    srt = np.take_along_axis(s, order, axis=1)
                    self.min_gap = min(self.min_gap, float((srt[:, kk - 1] - srt[:, kk]).min()))
        self.sel = {"idx": idx, "cnt": cnt, "sink": self.sink_ids() if cur["id"] > 0 else [],
                    "cur": self.current_ids()}
        return idx, cnt

    def kept_blocks(self, h: int, i: int) -> list[tuple[int, bool]]:
        """KEPT[h, i] = SINK u TOPK[h, i] u CUR as (global id, from_sink) pairs (BJ north_star:
        "keep top-k key blocks plus the always-kept sink and local blocks"; S8c-13/14/15).
        For c = 0 the sink lies inside CUR and is not listed twice."""
        sel = self.sel
        out = [(g, True) for g in sel["sink"]]
        out += [(int(g), False) for g in sel["idx"][h, i, :sel["cnt"][h, i]]]
        out += [(g, False) for g in sel["cur"]]
        return out

    # ----------------------------------------------------------------- step 3
    def sparse_attn(self, Q: np.ndarray, heads=None, qblocks=None, softmax_scale: float = 0.0):
        """o_n = sum_m softmax_m(q_n . k_m / sqrt(d)) v_m over all valid tokens m of KEPT[h, i]
        (natural exp, max-subtracted, S8c-20).  Returns O fp64 [n, H, d] and
        lse fp64 [H, n] (natural log); rows of (head, block) pairs not requested are NaN."""
        Q = np.asarray(Q, dtype=np.float64)
        cur = self.resident[-1]
        n = cur["n"]
        assert self.sel is not None, "select_blocks must run before sparse_attn"
        nqb = self.n_blocks(n)
        O = np.full((n, self.H, self.d), np.nan, dtype=np.float64)
        lse = np.full((self.H, n), np.nan, dtype=np.float64)
        heads = range(self.H) if heads is None else heads
        qblocks = range(nqb) if qblocks is None else qblocks
        for h in heads:
            for i in qblocks:
                lo, hi = i * self.B, min((i + 1) * self.B, n)
                q = Q[lo:hi, h, :]                                               # [r, d]
                ks, vs = [], []
                for g, from_sink in self.kept_blocks(h, i):
                    kr, vr = self.block_kv(g, from_sink)
                    ks.append(kr[:, h, :])
                    vs.append(vr[:, h, :])
                Kc = np.concatenate(ks, axis=0)                                  # [M, d]
                Vc = np.concatenate(vs, axis=0)
                logits = q @ Kc.T
                logits = logits * softmax_scale if softmax_scale else logits / math.sqrt(float(self.d))
                m = logits.max(axis=1, keepdims=True)
                p = np.exp(logits - m)
                l = p.sum(axis=1, keepdims=True)
                O[lo:hi, h, :] = (p @ Vc) / l
                lse[h, lo:hi] = (m + np.log(l))[:, 0]
        return O, lse

    # ------------------------------------------------------------ conveniences
    def kept_flop(self) -> int:
        """4 * d * sum over (h, i) of valid q rows x valid kept keys."""
        cur = self.resident[-1]
        n = cur["n"]
        total = 0
        for h in range(self.H):
            for i in range(self.n_blocks(n)):
                rows = min((i + 1) * self.B, n) - i * self.B
                keys = sum(self.block_kv(g, fs)[0].shape[0] for g, fs in self.kept_blocks(h, i))
                total += rows * keys
        return 4 * self.d * total
