"""Test harness: drive the same seeded chunk stream through the CUDA path (via the C ABI binding)
and through the fp64 oracle, and compare.  Test infrastructure only (imports `oracle/`)."""
from __future__ import annotations

import math

import numpy as np

import uf_workloads as wl
from oracle.uf_oracle import UFOracle

# BASELINE.json north_star: attention outputs within max-abs 2e-2 and mean-abs 2e-3 of the fp64 oracle
O_MAX_ABS = 2e-2
O_MEAN_ABS = 2e-3
# LSE has no tolerance in BASELINE.json; the bound is derived in DESIGN.md section 6 from the kernel's design: the
# row sum l adds the bf16-rounded probabilities (the numbers the P V MMA multiplies, which is what keeps O inside
# the BJ bound at every softmax scale), each within 2^-8 relative of its exact value (round-to-nearest, 8
# significant bits), so |l~/l - 1| <= 2^-8 and |dLSE| <= -ln(1 - 2^-8) = 3.92e-3; the degree-3 exp2 polynomial
# (7.5e-5), ex2.approx, the fp32 sum over <= 6e4 keys and log2f add < 1e-4.  Reached only by one-hot rows.
LSE_MAX_ABS = 4.1e-3


def bits_to_f64(bits: np.ndarray) -> np.ndarray:
    return wl.bf16_bits_to_f32(bits).astype(np.float64)


class CudaStream:
    """One ctx + torch device buffers; every step goes through the C ABI."""

    def __init__(self, w: wl.Workload, chunk_tokens_max: int | None = None, device: int = 0):
        import torch
        import paper_2606_09150_b200 as uf
        self.torch, self.uf, self.w = torch, uf, w
        self.dev = torch.device("cuda", device)
        self.nmax = w.chunk_tokens if chunk_tokens_max is None else chunk_tokens_max
        self.ctx = uf.uf_ctx_create(w.n_heads, w.head_dim, w.block, self.nmax, w.capacity_chunks,
                                    w.sink_blocks, w.k_min, device)
        self.stream = torch.cuda.current_stream(self.dev)

    def close(self):
        if self.ctx is not None:
            self.uf.uf_ctx_destroy(self.ctx)
            self.ctx = None

    def to_dev(self, bits: np.ndarray):
        t = self.torch.from_numpy(bits.view(np.int16)).to(self.dev)
        return t.view(self.torch.bfloat16)

    def step(self, Qb, Kb, Vb, topk_count=-1, topk_percent=-1, window=0, want_lse=True, impl=0, scale=0.0,
             fused_qkv=False):
        """append -> select -> attention for one chunk of bf16 bit arrays [n, H, d].
        fused_qkv: Q, K, V are the three slices of ONE [n, 3, H, d] tensor (token stride 3*H*d), the layout a
        fused QKV projection leaves them in, and O is written into a slice of a [n, 2, H, d] tensor.
        Returns dict(slot_map, idx, cnt, O (float32 [n,H,d]), lse (float32 [H,n]))."""
        torch, uf, w = self.torch, self.uf, self.w
        n, H, d = Qb.shape
        if fused_qkv:
            qkv = self.to_dev(np.ascontiguousarray(np.stack([Qb, Kb, Vb], axis=1)))      # [n, 3, H, d]
            q, k, v = qkv[:, 0], qkv[:, 1], qkv[:, 2]
            ts, hs = 3 * H * d, d
        else:
            q, k, v = self.to_dev(Qb), self.to_dev(Kb), self.to_dev(Vb)
            ts, hs = H * d, d
        uf.uf_kv_append(self.ctx, k, v, n, ts, hs, window, self.stream)
        slot_map = uf.uf_get_slot_map(self.ctx, w.capacity_chunks)
        n_cand, k_eff = uf.uf_query_topk(self.ctx, topk_count, topk_percent)
        nqb = -(-n // w.block)
        idx = torch.full((H, nqb, max(k_eff, 1)), -1, dtype=torch.int32, device=self.dev)
        cnt = torch.full((H, nqb), -1, dtype=torch.int32, device=self.dev)
        uf.uf_select_blocks(self.ctx, q, n, ts, hs, topk_count, topk_percent, idx, cnt, self.stream)
        if fused_qkv:
            o2 = torch.full((n, 2, H, d), float("nan"), dtype=torch.bfloat16, device=self.dev)
            o = o2[:, 1]
        else:
            o = torch.full((n, H, d), float("nan"), dtype=torch.bfloat16, device=self.dev)
        lse = torch.full((H, n), float("nan"), dtype=torch.float32, device=self.dev) if want_lse else None
        # shapes other than B = d = 128 have no tcgen05 kernel: the caller has to opt in to the CUDA-core kernel
        uf.uf_set_attn_impl(self.ctx, impl if (w.block == 128 and w.head_dim == 128) else 1)
        if fused_qkv:
            # attention takes one token stride for Q and O: O's [n, 2, H, d] slice has stride 2*H*d, so Q is
            # re-packed to that stride too (Q of the select call above kept the fused layout)
            q2 = torch.empty((n, 2, H, d), dtype=torch.bfloat16, device=self.dev)
            q2[:, 0] = q
            uf.uf_sparse_attn_fwd(self.ctx, q2[:, 0], o, lse, n, 2 * H * d, hs, scale, self.stream)
            torch.cuda.synchronize(self.dev)
            assert torch.isnan(o2[:, 0].float()).all(), "attention wrote outside its O slice"
        else:
            uf.uf_sparse_attn_fwd(self.ctx, q, o, lse, n, ts, hs, scale, self.stream)
        torch.cuda.synchronize(self.dev)
        return {
            "slot_map": slot_map, "n_cand": n_cand, "k_eff": k_eff,
            "idx": idx.cpu().numpy()[:, :, :k_eff], "cnt": cnt.cpu().numpy(),
            "O": o.float().cpu().numpy(), "lse": None if lse is None else lse.cpu().numpy(),
        }

    def cache_block(self, g: int, head: int):
        w = self.w
        kb = np.zeros((w.block, w.head_dim), dtype=np.uint16)
        vb = np.zeros((w.block, w.head_dim), dtype=np.uint16)
        self.uf.uf_get_cache_block(self.ctx, g, head, kb, vb, self.stream)
        return kb, vb

    def pooled_k(self, g: int, head: int):
        out = np.zeros(self.w.head_dim, dtype=np.float64)
        self.uf.uf_get_pooled_k(self.ctx, g, head, out, self.stream)
        return out


def make_oracle(w: wl.Workload, chunk_tokens_max: int | None = None) -> UFOracle:
    return UFOracle(w.n_heads, w.head_dim, w.block, w.chunk_tokens if chunk_tokens_max is None else chunk_tokens_max,
                    w.capacity_chunks, w.sink_blocks, w.k_min)


def oracle_step(orc: UFOracle, Qb, Kb, Vb, topk_count=-1, topk_percent=-1, window=0, heads=None, qblocks=None,
                scale=0.0, attn=True):
    Q, K, V = bits_to_f64(Qb), bits_to_f64(Kb), bits_to_f64(Vb)
    orc.kv_append(K, V, window)
    idx, cnt = orc.select_blocks(Q, topk_count, topk_percent)
    out = {"slot_map": orc.slot_map(), "idx": idx, "cnt": cnt, "min_gap": orc.min_gap}
    if attn:
        out["O"], out["lse"] = orc.sparse_attn(Q, heads=heads, qblocks=qblocks, softmax_scale=scale)
    return out


def compare_step(got: dict, ref: dict, where: str = "", o_max_abs: float = O_MAX_ABS):
    """Bit-exact slot map / indices / counts; O and LSE within tolerance on the rows the oracle computed."""
    assert got["slot_map"] == ref["slot_map"], f"{where} slot map {got['slot_map']} != {ref['slot_map']}"
    assert got["cnt"].shape == ref["cnt"].shape and np.array_equal(got["cnt"], ref["cnt"]), f"{where} counts differ"
    assert got["idx"].shape == ref["idx"].shape, f"{where} idx shape {got['idx'].shape} != {ref['idx'].shape}"
    if not np.array_equal(got["idx"], ref["idx"]):
        bad = np.argwhere(got["idx"] != ref["idx"])
        raise AssertionError(f"{where} selected block ids differ at {len(bad)} places, first {bad[0]} "
                             f"(oracle min top-k gap {ref.get('min_gap')})")
    if "O" in ref:
        mask = ~np.isnan(ref["O"])
        assert mask.any()
        assert not np.isnan(got["O"][mask]).any(), f"{where} CUDA output has NaN / unwritten rows"
        err = np.abs(got["O"].astype(np.float64)[mask] - ref["O"][mask])
        assert err.max() <= o_max_abs, f"{where} O max-abs {err.max():.3e} > {o_max_abs:.3e}"
        assert err.mean() <= O_MEAN_ABS, f"{where} O mean-abs {err.mean():.3e} > {O_MEAN_ABS}"
        if got.get("lse") is not None:
            lm = ~np.isnan(ref["lse"])
            lerr = np.abs(got["lse"].astype(np.float64)[lm] - ref["lse"][lm])
            assert lerr.max() <= LSE_MAX_ABS, f"{where} LSE max-abs {lerr.max():.3e} > {LSE_MAX_ABS}"
        return float(err.max()), float(err.mean())
    return None
