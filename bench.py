#!/usr/bin/env python
"""bench.py — measure the sparse causal chunk attention hot path (append -> select -> attention) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 1k|2k|wide|1k_stream] [--impl reference]

One "step" = one pass of the whole hot path over one chunk of synthetic
input shaped like BASELINE.json configs[1] (default; `--workload` picks another).  Prints ONE JSON line
(the contract is in DESIGN.md §"Measurement").  `value` = effective TFLOP/s counting only kept blocks,
over the whole step with inputs resident in HBM; `ms_per_step` = ms/chunk; `e2e` = the same through the
C ABI with pinned HOST buffers (H2D of Q,K,V and D2H of O inside the timed region); `roofline` = the
attention kernel alone against the measured bf16 tensor peak; `cpu_baseline` = the fp64 oracle timed on
this box's host cores on a bounded sample.  Multi-GPU = independent replicas (the path does
not shard by contract), one rank per GPU, max-over-ranks timing.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import uf_workloads as wl  # noqa: E402

PROFILE_TRAFFIC = os.path.join(ROOT, "profiles", "attn_dram_traffic.txt")
KERNEL_SOURCES = ["include/uf.h"] + ["paper_2606_09150_b200/csrc/" + f for f in (
    "uf_internal.h", "uf_sm100_ptx.h", "uf_api.cu", "uf_append.cu", "uf_fused_append.cu", "uf_select.cu", "uf_attn_generic.cu", "uf_attn_sm100.cu")]


def kernel_source_hash() -> str:
    """sha256 over the CUDA sources + the ABI header: ties an ncu capture under profiles/ to the code it profiled."""
    import hashlib
    h = hashlib.sha256()
    for rel in KERNEL_SOURCES:
        with open(os.path.join(ROOT, rel), "rb") as f:
            h.update(rel.encode() + b"\0" + f.read())
    return h.hexdigest()


def ncu_attn_dram_bytes(workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE uf_attn_sm100_kernel<false> launch, read from the
    committed summary of an `ncu --set full` capture (profiles/attn_dram_traffic.txt: `key: value` lines, the command
    that made it, and the sha256 of the sources it profiled).  None when there is no capture of this workload or when
    the sources have changed since: a stale number is not reported."""
    try:
        kv = {}
        for line in open(PROFILE_TRAFFIC):
            if ":" in line and not line.startswith("#"):
                k, v = line.split(":", 1)
                kv[k.strip()] = v.strip()
        if kv.get("source_sha256") != kernel_source_hash():
            return None, "capture is of other sources (profiles/attn_dram_traffic.txt): not reported"
        if workload not in kv:
            return None, "no capture of this workload"
        return float(kv[workload]), "ncu --set full capture, profiles/attn_dram_traffic.txt (sources match)"
    except OSError:
        return None, "no capture committed"


ATTN_IMPL = 0          # --attn-impl: which tcgen05 attention kernel uf_sparse_attn_fwd runs (uf_set_attn_impl)

METRIC = "effective TFLOP/s on kept blocks, sparse causal chunk attention step (ms/chunk in ms_per_step)"
UNIT = "TFLOP/s"


# --------------------------------------------------------------------------------------------------
def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"bf16_burst": float(p["bf16_tflops"]), "bf16_sustained": float(p["bf16_tflops_sustained"]),
                "hbm_gbs": float(p["hbm_gbs"]), "source": "measured (MEASURED_PEAKS.json)"}
    return {"bf16_burst": 1590.0, "bf16_sustained": 1400.0, "hbm_gbs": 6650.0,
            "source": "fallback (B200_PROFILING.md)"}


def kept_flop(w: wl.Workload, n_tok: int, idx: np.ndarray, sink_tok: int, prior_ntok: dict[int, int]) -> int:
    """4*d*sum over (h, i) of valid q rows x valid kept keys; bookkeeping from the index
    lists the library returned — no method arithmetic."""
    B, d, bpc = w.block, w.head_dim, -(-w.chunk_tokens // w.block)
    nqb = -(-n_tok // B)
    rows = np.minimum(B, n_tok - np.arange(nqb) * B).astype(np.int64)             # [nqb]
    if idx.size:
        cid, b = idx // bpc, idx % bpc
        ntok = np.vectorize(lambda c: prior_ntok[int(c)])(cid)
        keys_topk = np.minimum(B, ntok - b * B).astype(np.int64).sum(axis=2)      # [H, nqb]
    else:
        keys_topk = np.zeros((w.n_heads, nqb), dtype=np.int64)
    keys = keys_topk + sink_tok + n_tok
    return int(4 * d * (rows[None, :] * keys).sum())


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, device: int):
        self.rows, self.proc, self.device = [], None, device

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.device}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        hi = [x for x in sm if x >= 0.5 * max(sm)] or sm
        return {"sm_mhz": float(np.median(hi)), "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm)}


# --------------------------------------------------------------------------------------------------
def dist_setup(n_gpus: int):
    """One process per GPU under torchrun; returns (rank, world, local_rank)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        if not dist.is_initialized():
            backend = os.environ.get("UF_DIST_BACKEND", "nccl")
            dist.init_process_group(backend=backend)
    return rank, world, local


def aggregate_over_ranks(elapsed_ms: float, units: float, device=None):
    """Replicas only: time = max over ranks, units = sum over ranks (no data-path collective)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return elapsed_ms, units
    dev = device if device is not None else torch.device("cpu")
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


# --------------------------------------------------------------------------------------------------
_CHUNKS: dict = {}


def get_chunks(w: wl.Workload, ids):
    """Seeded chunks (bf16 bits) of a workload, generated on a thread pool and shared between workloads that have
    the same recipe (1k / 1k_stream / 1k_paper draw identical chunks: same grid, heads, amplitude, seeds)."""
    from concurrent.futures import ThreadPoolExecutor
    key = lambda c: (w.n_heads, w.head_dim, w.frames_per_chunk, w.grid_h, w.grid_w, w.amp, c)  # noqa: E731
    todo = [c for c in ids if key(c) not in _CHUNKS]
    if todo:
        with ThreadPoolExecutor(min(8, len(todo))) as ex:
            for c, ch in zip(todo, ex.map(lambda c: wl.make_chunk(w, c), todo)):
                _CHUNKS[key(c)] = ch
    return [_CHUNKS[key(c)] for c in ids]


def tile_sizes(w: wl.Workload) -> np.ndarray:
    """valid tokens of every tile of a chunk (paper-mask workloads), tile-major: bookkeeping for the FLOP count"""
    bt, bh, bw = w.tile
    vt = np.minimum(bt, w.frames_per_chunk - np.arange(w.tile_grid[0]) * bt)
    vh = np.minimum(bh, w.grid_h - np.arange(w.tile_grid[1]) * bh)
    vw = np.minimum(bw, w.grid_w - np.arange(w.tile_grid[2]) * bw)
    return (vt[:, None, None] * vh[None, :, None] * vw[None, None, :]).reshape(-1).astype(np.int64)


class HotPath:
    """The step bench.py times: uf_kv_append -> uf_select_blocks -> uf_sparse_attn_fwd via the C ABI
    (paper-mask workloads: a tiled ctx, uf_select_blocks_paper, chunks converted once by uf_tile_tokens)."""

    def __init__(self, w: wl.Workload, device: int, chunk_ids, pinned_host: bool, fused: bool = False):
        import torch
        import paper_2606_09150_b200 as uf
        self.torch, self.uf, self.w = torch, uf, w
        self.dev = torch.device("cuda", device)
        torch.cuda.set_device(self.dev)
        self.paper = w.tile is not None
        self.fused = fused          # NEXT-2: raw Q, K, V in; QK-norm + RoPE + append + pooling in one kernel
        self.H, self.d = w.n_heads, w.head_dim
        self.n = w.n_tiles * w.block if self.paper else w.chunk_tokens      # rows the library sees per chunk
        self.attn_impl = ATTN_IMPL
        self.ctx = uf.uf_ctx_create(w.n_heads, w.head_dim, w.block, self.n, w.capacity_chunks,
                                    0 if self.paper else w.sink_blocks, w.k_min, device)
        self.stream = torch.cuda.current_stream(self.dev)
        if self.attn_impl:
            uf.uf_set_attn_impl(self.ctx, self.attn_impl)
        if self.paper:
            uf.uf_ctx_set_tiling(self.ctx, w.frames_per_chunk, w.grid_h, w.grid_w, *w.tile, w.window)
        self.ts, self.hs = self.H * self.d, self.d
        self.host = []      # pinned host chunks (int16 views of bf16 bits), only for the e2e leg
        self.devc = []      # device-resident chunks
        for qb, kb, vb in get_chunks(w, chunk_ids):
            hq, hk, hv = (torch.from_numpy(x.view(np.int16)) for x in (qb, kb, vb))
            if pinned_host:
                hq, hk, hv = hq.pin_memory(), hk.pin_memory(), hv.pin_memory()
                self.host.append((hq, hk, hv))
            dq, dk, dv = (t.to(self.dev, non_blocking=True).view(torch.bfloat16) for t in (hq, hk, hv))
            if self.paper:
                tiled = []
                for t in (dq, dk, dv):
                    o = torch.empty((self.n, self.H, self.d), dtype=torch.bfloat16, device=self.dev)
                    uf.uf_tile_tokens(self.ctx, t, o, self.ts, self.hs, self.ts, self.hs, self.stream)
                    tiled.append(o)
                dq, dk, dv = tiled
            self.devc.append((dq, dk, dv))
        nqb = -(-self.n // w.block)
        kmax = max(1, w.capacity_chunks * w.bpc if not self.paper else w.capacity_chunks * w.n_tiles)
        self.idx = torch.zeros((self.H, nqb, kmax), dtype=torch.int32, device=self.dev)
        self.cnt = torch.zeros((self.H, nqb), dtype=torch.int32, device=self.dev)
        self.idx_stride = kmax
        self.o = torch.zeros((self.n, self.H, self.d), dtype=torch.bfloat16, device=self.dev)
        self.lse = torch.zeros((self.H, self.n), dtype=torch.float32, device=self.dev)
        if pinned_host:
            # e2e staging: two sets (double buffering): while step i computes, step i+1's inputs arrive and
            # step i-1's O leaves
            mk = lambda: torch.empty((self.n, self.H, self.d), dtype=torch.bfloat16, device=self.dev)  # noqa: E731
            self.stage = [tuple(mk() for _ in range(3)) for _ in range(2)]
            self.o_e2e = [mk() for _ in range(2)]
            self.o_host = [torch.empty((self.n, self.H, self.d), dtype=torch.bfloat16).pin_memory() for _ in range(2)]
            self.s_in, self.s_out = torch.cuda.Stream(self.dev), torch.cuda.Stream(self.dev)
            E = lambda: torch.cuda.Event()  # noqa: E731
            self.ev_in = [E(), E()]      # inputs of set b are on the device
            self.ev_free = [E(), E()]    # the step that read set b's inputs has finished
            self.ev_done = [E(), E()]    # O of set b is complete
            self.ev_out = [E(), E()]     # O of set b has been copied to the host
        if fused:
            self.max_pos = 1024
            cos, sin = wl.rope_tables(self.max_pos)
            gq, gk = wl.norm_weights(w)
            self.rope = tuple(torch.from_numpy(x).to(self.dev) for x in (cos, sin, gq, gk))
            self.q_rot = torch.zeros((self.n, self.H, self.d), dtype=torch.bfloat16, device=self.dev)
        self.e2e_no = 0
        self.step_no = 0
        torch.cuda.synchronize(self.dev)

    def close(self):
        self.uf.uf_ctx_destroy(self.ctx)

    def step(self, q, k, v, ev=None, ev_pre=None, window=0):
        """ev = (before attention, after attention); ev_pre = (before append, before select) for the
        per-call breakdown pass (not used inside the timed region)."""
        uf, w = self.uf, self.w
        if ev_pre is not None:
            ev_pre[0].record(self.stream)
        if self.fused:
            t0 = (self.step_no % 300) * w.frames_per_chunk
            uf.uf_qkv_rope_append(self.ctx, q, k, v, self.q_rot, self.n, self.ts, self.hs, self.ts, self.hs, *self.rope,
                                  self.max_pos, t0, w.grid_h, w.grid_w, wl.ROPE_AXIS_DIMS, 1e-6, window, self.stream)
            q = self.q_rot
        else:
            uf.uf_kv_append(self.ctx, k, v, self.n, self.ts, self.hs, window, self.stream)
        if ev_pre is not None:
            ev_pre[1].record(self.stream)
        if self.paper:
            uf.uf_select_blocks_paper(self.ctx, q, self.n, self.ts, self.hs, -1, w.rho_permille, self.idx,
                                      self.idx_stride, self.cnt, self.stream)
        else:
            uf.uf_select_blocks(self.ctx, q, self.n, self.ts, self.hs, w.topk_count, w.topk_percent,
                                self.idx, self.cnt, self.stream)
        if ev is not None:
            ev[0].record(self.stream)
        uf.uf_sparse_attn_fwd(self.ctx, q, self.o, self.lse, self.n, self.ts, self.hs, 0.0, self.stream)
        if ev is not None:
            ev[1].record(self.stream)
        self.step_no += 1

    def step_resident(self, ev=None, ev_pre=None):
        q, k, v = self.devc[self.step_no % len(self.devc)]
        self.step(q, k, v, ev, ev_pre)

    def step_e2e(self):
        """One end-to-end step through the C ABI: H2D of this step's Q,K,V from pinned host memory (copy stream),
        the three calls (compute stream), D2H of O to pinned host memory (output stream).  Consecutive steps are
        pipelined over two buffer sets the way a streaming caller would: the copies of neighbouring steps overlap
        this step's kernels, every step still moves all of its bytes inside the timed region."""
        torch, b = self.torch, self.e2e_no & 1
        hq, hk, hv = self.host[self.step_no % len(self.host)]
        sq, sk, sv = self.stage[b]
        with torch.cuda.stream(self.s_in):
            self.s_in.wait_event(self.ev_free[b])           # the step two back has finished with this set
            sq.view(torch.int16).copy_(hq, non_blocking=True)
            sk.view(torch.int16).copy_(hk, non_blocking=True)
            sv.view(torch.int16).copy_(hv, non_blocking=True)
            self.ev_in[b].record(self.s_in)
        self.stream.wait_event(self.ev_in[b])
        self.stream.wait_event(self.ev_out[b])              # O buffer b has left for the host
        o_saved, self.o = self.o, self.o_e2e[b]
        self.step(sq, sk, sv)
        self.o = o_saved
        self.ev_done[b].record(self.stream)
        self.ev_free[b].record(self.stream)
        with torch.cuda.stream(self.s_out):
            self.s_out.wait_event(self.ev_done[b])
            self.o_host[b].copy_(self.o_e2e[b], non_blocking=True)
            self.ev_out[b].record(self.s_out)
        self.e2e_no += 1

    def e2e_drain(self):
        """make the compute stream wait for every outstanding copy (called before the closing timing event)"""
        for b in range(2):
            self.stream.wait_event(self.ev_out[b])
            self.stream.wait_event(self.ev_in[b])

    def current_kept_flop(self):
        """FLOP of the step just run, from the returned index lists -> (kept FLOP, N candidates, k', extra)."""
        uf, w = self.uf, self.w
        self.torch.cuda.synchronize(self.dev)
        if self.paper:
            n_cand, k_eff = uf.uf_query_budget_paper(self.ctx, -1, w.rho_permille)
            idx, cnt = self.idx.cpu().numpy(), self.cnt.cpu().numpy()
            nv = tile_sizes(w)
            keys = np.where(idx >= 0, nv[np.maximum(idx, 0) % w.n_tiles], 0).sum(axis=2)          # [H, NB]
            flop = int(4 * self.d * (nv[None, :] * keys).sum())
            extra = {"mean_kept_blocks_per_row": float(cnt.mean()),
                     "tensor_pipe_tflop_incl_tile_padding": float(4 * self.d * 128 * 128 * cnt.sum()) / 1e12,
                     "tile_fill": float(nv.sum()) / float(nv.size * w.block)}
            return flop, n_cand, k_eff, extra
        n_cand, k_eff = uf.uf_query_topk(self.ctx, w.topk_count, w.topk_percent)
        nqb = self.idx.shape[1]
        idx = self.idx.cpu().numpy().reshape(-1)[: self.H * nqb * k_eff].reshape(self.H, nqb, k_eff)
        slot_map, _, newest = uf.uf_get_slot_map(self.ctx, w.capacity_chunks)
        prior = {c: self.n for c in slot_map if c >= 0}
        sink_tok = min(w.sink_blocks * w.block, self.n) if newest > 0 else 0
        return kept_flop(w, self.n, idx, sink_tok, prior), n_cand, k_eff, {}


def time_steps(hp: HotPath, steps: int, warmup: int, e2e: bool):
    torch = hp.torch
    for _ in range(warmup):
        hp.step_e2e() if e2e else hp.step_resident()
    if e2e:
        hp.e2e_drain()
    torch.cuda.synchronize(hp.dev)
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    attn_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    launches0 = hp.uf.uf_ctx_launch_count(hp.ctx)
    ev0.record(hp.stream)
    for i in range(steps):
        if e2e:
            hp.step_e2e()
        else:
            hp.step_resident(attn_ev[i])
    if e2e:
        hp.e2e_drain()
    ev1.record(hp.stream)
    torch.cuda.synchronize(hp.dev)
    barrier()
    total_ms = ev0.elapsed_time(ev1)
    attn_ms = None if e2e else float(np.mean([a.elapsed_time(b) for a, b in attn_ev]))
    launches = hp.uf.uf_ctx_launch_count(hp.ctx) - launches0
    return total_ms, attn_ms, launches


def time_sustained(hp: HotPath, seconds: float, ms_per_step_hint: float, device: int):
    """the default timed region is a ~70 ms burst; a streaming model runs for minutes.  Run the same
    device-resident step back to back for >= `seconds` of GPU time (the power cap pulls the SM clock down after
    ~50 ms) and report the whole-loop ms/step, the mean attention launch and the SM clock under load."""
    torch = hp.torch
    steps = int(math.ceil(seconds * 1.08 * 1e3 / ms_per_step_hint))
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    attn_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    torch.cuda.synchronize(hp.dev)
    with ClockSampler(device) as cs:
        ev0.record(hp.stream)
        for i in range(steps):
            hp.step_resident(attn_ev[i])
        ev1.record(hp.stream)
        torch.cuda.synchronize(hp.dev)
    total_ms = ev0.elapsed_time(ev1)
    attn = np.array([a.elapsed_time(b) for a, b in attn_ev])
    tail = attn[len(attn) // 2:]                                  # the second half: clocks have settled
    return {"steps": steps, "total_ms": total_ms, "attn_ms": float(attn.mean()), "attn_ms_second_half": float(tail.mean()),
            "attn_ms_first_10": float(attn[:10].mean()), "clocks": cs.summary()}


def call_breakdown(hp: HotPath, steps: int, hbm_gbs: float):
    """Separate pass after the timed region: CUDA events around each of the three C-ABI calls, and the
    HBM-roofline view of the two data-movement calls (algorithmic bytes of DESIGN.md 5.2 / 5.3)."""
    torch, w = hp.torch, hp.w
    E = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731
    evs = [(E(), E(), E(), E()) for _ in range(steps)]
    for e in evs:
        hp.step_resident(ev=(e[2], e[3]), ev_pre=(e[0], e[1]))
    torch.cuda.synchronize(hp.dev)
    app = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    sel = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    att = float(np.mean([e[2].elapsed_time(e[3]) for e in evs]))
    nhd2 = hp.n * hp.H * hp.d * 2
    nb = -(-hp.n // w.block)
    app_bytes = 4 * nhd2 + 8 * hp.H * hp.d * nb                       # read K,V + write both caches + pooled K
    if hp.fused:
        app_bytes = 6 * nhd2 + 2 * 8 * hp.H * hp.d * nb               # + read raw Q, write post-RoPE Q, pooled Q
    _, n_cand, k_eff, _ = hp.current_kept_flop()
    sel_bytes = nhd2 + 8 * hp.H * hp.d * (nb + n_cand) + 4 * hp.H * nb * (k_eff + 1)   # read Q, pooled Q/K, write ids
    if hp.fused:
        sel_bytes -= nhd2                                             # Q was pooled by the fused append
    return {
        "append": {"ms": app, "algorithmic_bytes": app_bytes, "achieved_gbs": app_bytes / app / 1e6,
                   "frac_of_hbm_peak": app_bytes / app / 1e6 / hbm_gbs},
        "select": {"ms": sel, "algorithmic_bytes": sel_bytes, "achieved_gbs": sel_bytes / sel / 1e6,
                   "frac_of_hbm_peak": sel_bytes / sel / 1e6 / hbm_gbs,
                   "note": ("1 kernel: fp64 score + exact top-k + pair merge (Q pooled by the fused append)" if hp.fused else
                            "2 kernels: pool Q (HBM-bound); fp64 score + exact threshold-search top-k + pair merge (latency/ALU-bound)")},
        "attention": {"ms": att},
        "hbm_peak_gbs": hbm_gbs,
    }


def stream_percentiles(hp: HotPath, repeats: int):
    """configs[3]: the 20-chunk rolling stream (per-chunk seeds 0..19) run `repeats` times after one untimed pass,
    CUDA events around every chunk; p50 / p99 over the steady-state chunks (c >= C), ramp-up chunks listed apart."""
    torch, w = hp.torch, hp.w
    per = []
    for rep in range(repeats + 1):
        hp.uf.uf_ctx_reset(hp.ctx, hp.stream)
        hp.step_no = 0
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(w.n_stream_chunks)]
        for c in range(w.n_stream_chunks):
            evs[c][0].record(hp.stream)
            hp.step_resident()
            evs[c][1].record(hp.stream)
        torch.cuda.synchronize(hp.dev)
        if rep:
            per.append([a.elapsed_time(b) for a, b in evs])
    per = np.asarray(per)
    steady = per[:, w.capacity_chunks:].reshape(-1)
    return {"p50_ms": float(np.percentile(steady, 50)), "p99_ms": float(np.percentile(steady, 99)),
            "mean_ms": float(steady.mean()), "max_ms": float(steady.max()), "steady_state_chunks_timed": int(steady.size),
            "rampup_ms": [float(x) for x in per[:, :w.capacity_chunks].mean(axis=0)], "repeats": repeats,
            "chunks_per_stream": w.n_stream_chunks}


def window_policy_curve(hp: HotPath):
    """NEXT-3: the 20-chunk rolling stream under each cache-window policy (uf_next_window feeding uf_kv_append's
    window_chunks): mean ms/chunk over chunks c >= C and mean resident K+V cache bytes, against the fixed window."""
    torch, uf, w = hp.torch, hp.uf, hp.w
    slot = 2 * hp.H * w.bpc * w.block * hp.d * 2
    policies = {
        "fixed": dict(kind=uf.UF_WIN_FIXED),
        "position(warm=3,compact=2)": dict(kind=uf.UF_WIN_POSITION, warm_chunks=3, compact_window=2),
        "memory(budget=2 slots)": dict(kind=uf.UF_WIN_MEMORY, budget_bytes=2 * slot),
        "content(min_share=300 permille,compact=1)": dict(kind=uf.UF_WIN_CONTENT, compact_window=1, min_share_permille=300),
    }
    out = {}
    for name, kw in policies.items():
        per, res, wins = [], [], []
        for rep in range(2):
            uf.uf_ctx_reset(hp.ctx, hp.stream)
            hp.step_no = 0
            evs = []
            for c in range(w.n_stream_chunks):
                W = uf.uf_next_window(hp.ctx, stream=hp.stream, **kw)       # content: one stream sync per chunk
                e = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                e[0].record(hp.stream)
                q, k, v = hp.devc[hp.step_no % len(hp.devc)]
                hp.step(q, k, v, window=W)
                e[1].record(hp.stream)
                evs.append(e)
                if rep:
                    wins.append(W)
                    res.append(uf.uf_get_slot_map(hp.ctx, w.capacity_chunks)[1])
            torch.cuda.synchronize(hp.dev)
            if rep:
                per = [a.elapsed_time(b) for a, b in evs]
        steady = per[w.capacity_chunks:]
        out[name] = {"ms_per_chunk_mean": float(np.mean(steady)), "resident_chunks_mean": float(np.mean(res[w.capacity_chunks:])),
                     "cache_bytes_mean": float(np.mean(res[w.capacity_chunks:])) * slot, "windows": wins}
    return out


# --------------------------------------------------------------------------------------------------
def blas_threads() -> int:
    try:
        from threadpoolctl import threadpool_info
        return max([int(x.get("num_threads", 1)) for x in threadpool_info()] or [1])
    except Exception:
        return 0


def cpu_oracle_sample(w: wl.Workload, n_random: int = 64, budget_s: float = 25.0):
    """The fp64 oracle as it stands, on this box's host cores: append and the FULL selection of
    the timed chunk, then attention on a seeded sample of (head, query-block) pairs: block 0, the ragged last block
    and `n_random` random pairs (cut short after `budget_s` seconds of attention, never below the two fixed pairs).
    Returns a dict with the measured seconds and the extrapolation to the full chunk by kept-FLOP ratio."""
    from oracle.uf_oracle import UFOracle
    cores = len(os.sched_getaffinity(0))
    orc = UFOracle(w.n_heads, w.head_dim, w.block, w.chunk_tokens, w.capacity_chunks, w.sink_blocks, w.k_min)
    f64 = lambda b: wl.bf16_bits_to_f32(b).astype(np.float64)  # noqa: E731
    chunks = get_chunks(w, range(w.prior_chunks + 1))
    for c in range(w.prior_chunks):
        _, kb, vb = chunks[c]
        orc.kv_append(f64(kb), f64(vb))
    qb, kb, vb = chunks[w.prior_chunks]
    Q, K, V = f64(qb), f64(kb), f64(vb)
    t0 = time.perf_counter()
    orc.kv_append(K, V)
    t_app = time.perf_counter() - t0
    t0 = time.perf_counter()
    orc.select_blocks(Q, w.topk_count, w.topk_percent)
    t_sel = time.perf_counter() - t0
    rng = np.random.default_rng(0)
    nqb = w.bpc
    pairs = [(0, 0), (w.n_heads - 1, nqb - 1)]
    pairs += [(int(rng.integers(0, w.n_heads)), int(rng.integers(0, nqb))) for _ in range(n_random)]

    def pair_flop(h, i):
        rows = min((i + 1) * w.block, w.chunk_tokens) - i * w.block
        keys = sum(orc.block_kv(g, fs)[0].shape[0] for g, fs in orc.kept_blocks(h, i))
        return 4 * w.head_dim * rows * keys

    t_attn, flop, done = 0.0, 0, 0
    for h, i in pairs:
        if done >= 2 and t_attn > budget_s:
            break
        t0 = time.perf_counter()
        orc.sparse_attn(Q, heads=[h], qblocks=[i])
        t_attn += time.perf_counter() - t0
        flop += pair_flop(h, i)
        done += 1
    total_flop = orc.kept_flop()
    attn_full = t_attn * total_flop / flop
    return {
        "value": flop / t_attn / 1e12, "unit": UNIT, "cores": cores, "kind": "oracle", "blas_threads": blas_threads(),
        "append_s": t_app, "select_full_s": t_sel, "attention_sample_s": t_attn, "attention_sample_pairs": done,
        "attention_pairs_total": w.n_heads * nqb, "attention_sample_flop": flop, "chunk_kept_flop": total_flop,
        "attention_s_per_chunk_extrapolated": attn_full,
        "chunk_s_extrapolated": t_app + t_sel + attn_full,
        "sample": (f"oracle/uf_oracle.py (NumPy fp64) on workload {w.name}: append and full selection timed in full; "
                   f"attention on {done} (head, query-block) pairs = block 0, the ragged last block and "
                   f"{max(done - 2, 0)} seeded random pairs of {w.n_heads * nqb}; value = sampled kept FLOP / attention "
                   f"seconds; *_extrapolated = sample time x (kept FLOP of the chunk / kept FLOP of the sample) — an "
                   f"extrapolation, not a measurement"),
    }


def run_reference(args, w):
    """--impl reference: the oracle timed on host cores; rank 0 only.  Each step = one bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    steps = max(1, min(args.steps, 3))
    for _ in range(1 if args.warmup >= 1 else 0):
        cpu_oracle_sample(w, n_random=2, budget_s=2.0)
    runs = [cpu_oracle_sample(w, n_random=16, budget_s=8.0) for _ in range(steps)]
    value = float(np.mean([r["value"] for r in runs]))
    t_all = float(np.sum([r["attention_sample_s"] for r in runs]))
    cb = dict(runs[-1])
    cb["value"] = value
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": 1, "ms_per_step": 1e3 * t_all / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "note": "each step = a bounded sample of the workload (see cpu_baseline.sample)"},
        "cpu_baseline": cb,
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------
# causal memory network streaming step (include/uf_cmn.h)
CMN_METRIC = "effective TFLOP/s of the causal memory network streaming step (ms/chunk in ms_per_step)"


def cmn_cpu_oracle(cw, budget_frames: int = 1):
    """the oracle's streaming step timed on host cores on a bounded crop of the workload (same network, same
    weights, a 20 x 36 grid, one frame): a reported baseline, TFLOP/s by the definition's FLOP count"""
    from oracle import uf_causal_mem as cm
    crop = wl.scaled_cmn(cw, cw.name + "_crop20x36", height=20, width=36, frames_per_chunk=budget_frames)
    cfg = cm.CmnConfig(crop.in_ch, crop.out_ch, tuple(crop.stage_channels), crop.n_blocks,
                       tuple(crop.spatial_factors), tuple(crop.temporal_factors))
    wt = {k: v.astype(np.float64) for k, v in wl.cmn_weights(crop).items()}
    z = wl.bf16_bits_to_f32(wl.cmn_frames(crop, 0)).astype(np.float64)
    st = cm.CausalMemStream(cfg, wt)
    t0 = time.perf_counter()
    st.step(z)
    dt = time.perf_counter() - t0
    fl = cm.flop_count(cfg, crop.height, crop.width, budget_frames)
    return {"value": fl / dt / 1e12, "unit": UNIT, "cores": len(os.sched_getaffinity(0)), "kind": "oracle",
            "blas_threads": blas_threads(), "seconds": dt,
            "sample": f"oracle/uf_causal_mem.py CausalMemStream.step (NumPy fp64) on {budget_frames} frame(s) of a "
                      f"{crop.height} x {crop.width} crop of workload {cw.name} ({fl / 1e9:.1f} GFLOP)"}


def measure_cmn(cw, device, steps, warmup, with_e2e=True, with_cpu=True):
    """device-resident steps of uf_cmn_step over a rotating set of chunks (+ e2e with pinned host frames in and the
    output back per step); the whole step is launches of ONE kernel template, so the roofline object is the step's"""
    import torch
    import paper_2606_09150_b200 as uf
    dev = torch.device("cuda", device)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream(dev)
    F = cw.frames_per_chunk
    rs, ts = int(np.prod(cw.spatial_factors)), int(np.prod(cw.temporal_factors))
    net = uf.uf_cmn_create(cw.in_ch, cw.out_ch, cw.stage_channels, cw.n_blocks, cw.spatial_factors,
                           cw.temporal_factors, cw.height, cw.width, F, device)
    try:
        wt = wl.cmn_weights(cw)
        for i in range(uf.uf_cmn_n_params(net)):
            name, shape, has_bias = uf.uf_cmn_param_info(net, i)
            w = np.ascontiguousarray(wl.f32_to_bf16_bits(wt[name]).reshape(shape))
            uf.uf_cmn_set_param(net, name, w, np.ascontiguousarray(wt[name + ".b"]) if has_bias else None)
        n_rot = 4
        host = [torch.from_numpy(wl.cmn_frames(cw, c).view(np.int16)).pin_memory() for c in range(n_rot)]
        z_dev = [h.to(dev).view(torch.bfloat16) for h in host]
        out_shape = (F * ts, cw.height * rs, cw.width * rs, cw.out_ch)
        out = torch.empty(out_shape, dtype=torch.bfloat16, device=dev)
        out_host = torch.empty(out_shape, dtype=torch.bfloat16).pin_memory()
        z_stage = torch.empty_like(z_dev[0])
        uf.uf_cmn_reset(net, stream)

        def run(n, e2e):
            for i in range(n):
                if e2e:
                    z_stage.view(torch.int16).copy_(host[i % n_rot], non_blocking=True)
                    uf.uf_cmn_step(net, z_stage, F, out, stream)
                    out_host.copy_(out, non_blocking=True)
                else:
                    uf.uf_cmn_step(net, z_dev[i % n_rot], F, out, stream)

        def timed(n, e2e):
            run(warmup, e2e)
            torch.cuda.synchronize(dev)
            barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            l0 = uf.uf_cmn_launches(net)
            e0.record(stream)
            run(n, e2e)
            e1.record(stream)
            torch.cuda.synchronize(dev)
            barrier()
            return e0.elapsed_time(e1), uf.uf_cmn_launches(net) - l0

        with ClockSampler(device) as cs:
            total_ms, launches = timed(steps, False)
        flop = uf.uf_cmn_flops(net, F)
        m = {"total_ms": total_ms, "steps": steps, "flop": flop, "launches": launches, "clocks": cs.summary(),
             "device_bytes": uf.uf_cmn_device_bytes(net), "n_layers": uf.uf_cmn_n_layers(net),
             "h2d": int(host[0].numel() * 2), "d2h": int(out.numel() * 2)}
        if with_e2e:
            m["e2e_ms"], _ = timed(steps, True)
        if with_cpu:
            m["cpu"] = cmn_cpu_oracle(cw)
        return m
    finally:
        uf.uf_cmn_destroy(net)


def cmn_layer_costs(cw):
    """[(layer, FLOP, algorithmic bytes)] of one uf_cmn_step over a chunk, from the network's shapes (bookkeeping only):
    bytes = input activations (+ one memory frame for a block's Conv1, R-41) + weights + output activations, all bf16;
    FLOP = 2 * multiply-adds with the real channel counts (the definition's count, oracle flop_count's)."""
    F, px = cw.frames_per_chunk, cw.height * cw.width
    ch = list(cw.stage_channels)
    n_stages = len(cw.spatial_factors)
    out = []

    def add(name, cin, cout, taps, in_frames=None, extra_in=0):
        act_in = (F if in_frames is None else in_frames) * px * cin * 2 + extra_in
        out.append((name, 2 * F * px * cout * cin * taps, act_in + cout * cin * taps * 2 + F * px * cout * 2))

    add("in", cw.in_ch, ch[0], 9)
    for s in range(n_stages):
        C = ch[s]
        for b in range(cw.n_blocks):
            add(f"s{s}.b{b}.c1", 2 * C, C, 9, in_frames=0, extra_in=(F + 1) * px * C * 2)     # h and h shifted by a frame
            add(f"s{s}.b{b}.c2", C, C, 9)
            out.append((f"s{s}.b{b}.c3+skip", 2 * F * px * C * C * 10, 3 * F * px * C * 2 + C * C * 10 * 2))
        r, t = cw.spatial_factors[s], cw.temporal_factors[s]
        add(f"s{s}.up", C, C * r * r, 9)
        px *= r * r
        if t > 1:
            add(f"s{s}.texp", C, C * t, 1)
            F *= t
        add(f"s{s}.ch", C, ch[s + 1] if s + 1 < len(ch) else C, 1)
    add("out", ch[n_stages] if n_stages < len(ch) else ch[n_stages - 1], cw.out_ch, 9)
    return out


def cmn_mixed_roofline(cw, ms_per_step, peaks):
    """a step of many layers has no single bound.  floor = sum over layers of max(FLOP / bf16 peak,
    bytes / HBM peak): what the step would take if every layer ran at whichever of its two rooflines is lower."""
    rows = cmn_layer_costs(cw)
    t_tensor = [f / (peaks["bf16_burst"] * 1e12) * 1e3 for _, f, _ in rows]
    t_hbm = [b / (peaks["hbm_gbs"] * 1e9) * 1e3 for _, _, b in rows]
    floor = sum(max(a, b) for a, b in zip(t_tensor, t_hbm))
    return {"floor_ms": floor, "frac": floor / ms_per_step, "tensor_only_ms": sum(t_tensor), "hbm_only_ms": sum(t_hbm),
            "hbm_bound_layers": [n for (n, _, _), a, b in zip(rows, t_tensor, t_hbm) if b > a],
            "algorithmic_bytes_per_step": int(sum(b for _, _, b in rows)), "flop_per_step": int(sum(f for _, f, _ in rows)),
            "peaks": {"bf16_tflops": peaks["bf16_burst"], "hbm_gbs": peaks["hbm_gbs"]}}


def cmn_entry(cw, m, peaks):
    steps = m["steps"]
    t = m["flop"] * steps / (m["total_ms"] * 1e-3) / 1e12
    e = {"workload": f"{cw.name} (PAPER.md:345-347 network: widths {list(cw.stage_channels)}, {cw.n_blocks} blocks/stage, "
                     f"spatial {list(cw.spatial_factors)}, temporal {list(cw.temporal_factors)}; input {cw.frames_per_chunk} x "
                     f"{cw.height} x {cw.width} x {cw.in_ch} per chunk)",
         "metric": CMN_METRIC, "steps": steps, "ms_per_step": m["total_ms"] / steps, "value": t, "unit": UNIT,
         "tflop_per_step": m["flop"] / 1e12, "gpu_launches": m["launches"], "layers_per_step": m["n_layers"],
         "ctx_device_bytes": m["device_bytes"], "clocks": m["clocks"],
         "roofline": {"kernel": "uf_cmn_conv_kernel (every layer of the step is a launch of it)", "bound": "tensor",
                      "achieved": t, "peak": peaks["bf16_burst"], "unit": UNIT, "frac": t / peaks["bf16_burst"],
                      "traffic": None, "peak_source": peaks["source"] + ", bf16 burst",
                      "algorithmic_flop_per_step": m["flop"],
                      "note": "FLOP by the definition (real channel counts); time = the whole step incl. launch gaps"}}
    e["roofline_mixed"] = cmn_mixed_roofline(cw, m["total_ms"] / steps, peaks)
    assert e["roofline_mixed"]["flop_per_step"] == m["flop"], (e["roofline_mixed"]["flop_per_step"], m["flop"])
    if "e2e_ms" in m:
        e["e2e"] = {"value": m["flop"] * steps / (m["e2e_ms"] * 1e-3) / 1e12, "unit": UNIT,
                    "ms_per_step": m["e2e_ms"] / steps, "h2d_bytes_per_step": m["h2d"], "d2h_bytes_per_step": m["d2h"]}
    if "cpu" in m:
        e["cpu_baseline"] = m["cpu"]
    return e


# --------------------------------------------------------------------------------------------------
def measure_workload(w, device, steps, warmup, with_e2e=True, stream_repeats=5, fused=False, sustained_s=0.0):
    """device-resident steps (+ attention events), per-call breakdown, optional e2e leg, optional rolling stream"""
    ids = range(w.n_stream_chunks) if w.n_stream_chunks else range(w.capacity_chunks + 1)
    hp = HotPath(w, device, ids, pinned_host=with_e2e, fused=fused)
    try:
        # reach steady state (chunk 0 evicted, all slots used) before anything is timed
        for _ in range(w.capacity_chunks + 1):
            hp.step_resident()
        with ClockSampler(device) as cs:
            total_ms, attn_ms, launches = time_steps(hp, steps, warmup, e2e=False)
        flop, n_cand, k_eff, extra = hp.current_kept_flop()
        out = {"total_ms": total_ms, "attn_ms": attn_ms, "launches": launches, "flop": flop, "n_cand": n_cand,
               "k_eff": k_eff, "clocks": cs.summary(), "device_bytes": hp.uf.uf_ctx_device_bytes(hp.ctx),
               "extra": extra, "steps": steps}
        out["calls"] = call_breakdown(hp, min(steps, 10), load_peaks()["hbm_gbs"])
        if sustained_s > 0:
            out["sustained"] = time_sustained(hp, sustained_s, total_ms / steps, device)
        out["h2d"] = 3 * hp.n * hp.H * hp.d * 2
        out["d2h"] = hp.n * hp.H * hp.d * 2
        if with_e2e:
            e2e_ms, _, _ = time_steps(hp, steps, min(warmup, 3), e2e=True)
            out["e2e_ms"] = e2e_ms
        if w.n_stream_chunks:
            out["stream"] = stream_percentiles(hp, repeats=stream_repeats)
            out["stream"]["window_policies"] = window_policy_curve(hp)
        return out
    finally:
        hp.close()


def roofline_obj(w, m, peaks):
    t = m["flop"] / (m["attn_ms"] * 1e-3) / 1e12
    traffic, src = ncu_attn_dram_bytes(w.name)
    return {
        "kernel": "uf_attn_sm100_kernel", "bound": "tensor", "achieved": t, "peak": peaks["bf16_burst"],
        "unit": "TFLOP/s", "frac": t / peaks["bf16_burst"], "traffic": traffic, "traffic_source": src,
        "peak_source": peaks["source"] + ", bf16 burst (the kernel is timed in a short burst; the >= 2 s loop under "
                       "config.sustained is the one divided by the sustained peak)",
        "algorithmic_flop_per_launch": m["flop"], "launch_ms": m["attn_ms"],
    }


def also_entry(w, m, peaks):
    """one secondary workload under `also`: the same quantities as the main line, compact"""
    steps = m["steps"]
    e = {"workload": w.name, "steps": steps, "ms_per_step": m["total_ms"] / steps, "attn_ms": m["attn_ms"],
         "kept_tflop_per_step": m["flop"] / 1e12, "value": m["flop"] * steps / (m["total_ms"] * 1e-3) / 1e12,
         "unit": UNIT, "k_eff": m["k_eff"], "n_cand": m["n_cand"], "gpu_launches": m["launches"],
         "roofline": roofline_obj(w, m, peaks), "calls": m["calls"], "clocks": m["clocks"]}
    if "e2e_ms" in m:
        e["e2e"] = {"value": m["flop"] * steps / (m["e2e_ms"] * 1e-3) / 1e12, "unit": UNIT,
                    "ms_per_step": m["e2e_ms"] / steps, "h2d_bytes_per_step": m["h2d"], "d2h_bytes_per_step": m["d2h"]}
    if "stream" in m:
        e["stream"] = m["stream"]
    if m["extra"]:
        e["paper_mask"] = m["extra"]
    return e


def cmn_main(args):
    """--workload cmn_*: the causal memory network step as its own line (used for its ncu captures)"""
    import torch
    cw = wl.CMN_CONFIGS[args.workload]
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) == 0:
            cb = cmn_cpu_oracle(cw)
            print(json.dumps({"impl": "reference", "metric": CMN_METRIC, "value": cb["value"], "unit": UNIT,
                              "n_gpus": args.gpus, "steps": 1, "warmup": 0, "ms_per_step": 1e3 * cb["seconds"],
                              "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                              "data": "synthetic", "config": {"workload": cw.name}, "cpu_baseline": cb,
                              "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0,
                                      "d2h_bytes_per_step": 0}, "gpu_launches": 0}), flush=True)
        return
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    rank, world, local = dist_setup(args.gpus)
    device = local if world > 1 else 0
    peaks = load_peaks()
    m = measure_cmn(cw, device, args.steps, max(3, args.warmup), with_cpu=(rank == 0 and not args.no_cpu_baseline))
    e = cmn_entry(cw, m, peaks)
    dev = torch.device("cuda", device)
    total_ms, units = aggregate_over_ranks(m["total_ms"], float(m["flop"]) * args.steps, dev)
    line = {"metric": CMN_METRIC, "value": units / (total_ms * 1e-3) / 1e12, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": e["workload"], "step": "uf_cmn_step (every layer a tcgen05 implicit-GEMM launch)",
                       "tflop_per_step": e["tflop_per_step"], "l2": "activations of a step exceed L2 only at the "
                       "decoder sizes; inputs rotate over 4 chunks", "parallelism": "replicas only" if world > 1 else "single GPU"},
            "e2e": e.get("e2e"), "gpu_launches": e["gpu_launches"], "clocks": e["clocks"], "roofline": e["roofline"]}
    if "cpu_baseline" in e:
        line["cpu_baseline"] = e["cpu_baseline"]
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="1k", choices=["1k", "2k", "wide", "1k_stream", "1k_paper", "2k_paper", "1k_paper_native",
                                                         "cmn_upsampler_1k", "cmn_decoder_crop", "cmn_decoder_1k"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sustained-seconds", type=float, default=2.0,
                    help="length of the back-to-back resident loop reported under config.sustained (0 = skip; N = 1 only)")
    ap.add_argument("--attn-impl", type=int, default=0, choices=[0, 2],
                    help="uf_set_attn_impl: 0 = the default tcgen05 attention kernel, 2 = the other tcgen05 variant")
    ap.add_argument("--no-also", action="store_true", help="skip the secondary workloads (2k, wide, 1k_stream, paper-mask variants)")
    ap.add_argument("--also", default="2k,1k_stream,wide,1k_paper,2k_paper,1k_paper_native,1k_fused,2k_fused,cmn_upsampler_1k,cmn_decoder_crop,cmn_decoder_1k",
                    help="comma list of secondary workloads (x_fused = workload x through uf_qkv_rope_append)")
    args = ap.parse_args()
    global ATTN_IMPL
    ATTN_IMPL = args.attn_impl
    if args.workload.startswith("cmn_"):
        cmn_main(args)
        return
    w = wl.CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, wl.CONFIGS["1k"] if w.tile else w)
        return
    warmup = max(3, args.warmup)

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    rank, world, local = dist_setup(args.gpus)
    device = local if world > 1 else 0
    peaks = load_peaks()

    m = measure_workload(w, device, args.steps, warmup, sustained_s=args.sustained_seconds if world == 1 else 0.0)
    dev = torch.device("cuda", device)
    total_ms, units = aggregate_over_ranks(m["total_ms"], float(m["flop"]) * args.steps, dev)
    e2e_ms, _ = aggregate_over_ranks(m["e2e_ms"], 0.0, dev)
    n_ranks = world
    value = units / (total_ms * 1e-3) / 1e12
    e2e_value = units / (e2e_ms * 1e-3) / 1e12

    if w.tile:
        what = (f"paper mask: tiles {w.tile}, window {w.window}, rho {w.rho_permille / 1000:.2f} -> tau_k {m['k_eff']} "
                f"of {m['n_cand']} blocks in the causal mask")
    else:
        what = f"keep {w.topk_percent}% of {m['n_cand']} cache blocks = {m['k_eff']}"
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": n_ranks, "steps": args.steps, "warmup": warmup,
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": {
            "workload": f"{w.name} (BASELINE.json configs: {w.n_heads} heads x {w.head_dim}, chunk {w.chunk_tokens} tokens, "
                        f"block {w.block}, capacity {w.capacity_chunks} chunks{'' if w.tile else ' + sink'}, {what})",
            "step": "uf_kv_append -> uf_select_blocks -> uf_sparse_attn_fwd, steady-state rolling cache",
            "kept_tflop_per_step": m["flop"] / 1e12,
            "l2": "inputs larger than L2 (Q,K,V 3 x %.0f MB + cache %.0f MB per step; no explicit flush)" % (
                m["d2h"] / 1e6, 2 * m["d2h"] * w.capacity_chunks / 1e6),
            "parallelism": "replicas only" if n_ranks > 1 else "single GPU",
            "attn_ms": m["attn_ms"], "append_select_ms": total_ms / args.steps - m["attn_ms"] if n_ranks == 1 else None,
            "ctx_device_bytes": m["device_bytes"],
            "e2e_note": "the e2e leg ships Q, K and V of every chunk from pinned host memory and O back (PCIe-bound: "
                        "h2d + d2h bytes below); in the paper's pipeline they are produced and consumed on the device "
                        "(P:1111), so e2e vs device ms/step is the link, not library overhead",
        },
        "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms / args.steps,
                "h2d_bytes_per_step": m["h2d"], "d2h_bytes_per_step": m["d2h"]},
        "gpu_launches": m["launches"],
        "clocks": m["clocks"],
        "roofline": roofline_obj(w, m, peaks),
        "calls": m["calls"],
    }
    if m["extra"]:
        line["config"]["paper_mask"] = m["extra"]
    if "stream" in m:
        line["stream"] = m["stream"]
    if "sustained" in m:
        # the same resident step, back to back for >= 2 s: clocks settle under the power cap, so THIS leg is the one
        # that may be divided by the sustained cuBLAS peak (MEASURED_PEAKS.json bf16_tflops_sustained)
        su = m["sustained"]
        t_attn = m["flop"] / (su["attn_ms_second_half"] * 1e-3) / 1e12
        line["config"]["sustained"] = {
            "seconds": su["total_ms"] * 1e-3, "steps": su["steps"], "ms_per_step": su["total_ms"] / su["steps"],
            "value": m["flop"] * su["steps"] / (su["total_ms"] * 1e-3) / 1e12,
            "attn_ms": su["attn_ms"], "attn_ms_first_10": su["attn_ms_first_10"],
            "attn_ms_second_half": su["attn_ms_second_half"], "attn_tflops_second_half": t_attn,
            "sustained_peak": peaks["bf16_sustained"], "frac_of_sustained_peak": t_attn / peaks["bf16_sustained"],
            "frac_of_burst_peak": t_attn / peaks["bf16_burst"],
            "sm_mhz_median": su["clocks"].get("sm_mhz"), "reasons": su["clocks"].get("reasons")}
    if rank == 0 and n_ranks == 1 and not args.no_also and args.workload == "1k":
        line["also"] = {}
        for name in [x for x in args.also.split(",") if x]:
            if name.startswith("cmn_"):
                cw = wl.CMN_CONFIGS[name]
                line["also"][name] = cmn_entry(cw, measure_cmn(cw, device, max(3, args.steps // 2), 3,
                                                               with_cpu=not args.no_cpu_baseline), peaks)
                ce = line["also"][name]
                line["config"][name] = {"steps": ce["steps"], "ms_per_step": ce["ms_per_step"], "value": ce["value"],
                                        "frac_burst": ce["roofline"]["frac"], "bound": ce["roofline"]["bound"],
                                        "mixed_floor_ms": ce["roofline_mixed"]["floor_ms"],
                                        "frac_mixed": ce["roofline_mixed"]["frac"],
                                        "hbm_bound_layers": ce["roofline_mixed"]["hbm_bound_layers"],
                                        "ctx_device_bytes": ce["ctx_device_bytes"]}
                continue
            fused = name.endswith("_fused")
            w2 = wl.CONFIGS[name[:-6] if fused else name]
            steps2 = max(3, args.steps // 2)
            m2 = measure_workload(w2, device, steps2, 3, with_e2e=(name == "2k"), fused=fused)
            line["also"][name] = also_entry(w2, m2, peaks)
            if name == "2k":
                # BASELINE.json's metric is quoted "at 1K/2K": the 2K half (configs[2]) in the kept part
                e2 = line["also"][name]
                line["config"]["k2"] = {
                    "workload": "2k (BASELINE.json configs[2])", "steps": e2["steps"], "ms_per_step": e2["ms_per_step"],
                    "attn_ms": e2["attn_ms"], "value": e2["value"], "kept_tflop_per_step": e2["kept_tflop_per_step"],
                    "frac_burst": e2["roofline"]["frac"], "traffic": e2["roofline"]["traffic"],
                    "e2e_ms_per_step": e2.get("e2e", {}).get("ms_per_step")}
            if fused:
                line["also"][name]["step"] = ("uf_qkv_rope_append (QK-norm + 3-D RoPE + append + pooled K, Q) -> "
                                              "uf_select_blocks (score + top-k only) -> uf_sparse_attn_fwd")
    if rank == 0 and n_ranks == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_oracle_sample(wl.CONFIGS["1k"] if w.tile else w)
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
