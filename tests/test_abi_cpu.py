"""CPU-side tests of the boundary: libuf.so builds, loads without a GPU, exports every symbol that
include/uf.h declares, and its host logic (cache slot policy, top-k budget, argument checks) agrees
with the oracle's state machine.  No compute call is made (there is no GPU here)."""
from __future__ import annotations

import os
import re

import numpy as np
import pytest

import paper_2606_09150_b200 as uf
from paper_2606_09150_b200 import binding
from oracle.uf_oracle import UFOracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    uf.build()
    return uf.load_library()


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "uf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(uf_[a-z_0-9]+)\s*\(", hdr)))
    assert declared == sorted(binding.SYMBOLS), (declared, sorted(binding.SYMBOLS))
    for name in declared:
        assert hasattr(lib, name), f"libuf.so does not export {name}"
    assert "sm_100a" in uf.uf_version()


def test_library_exports_every_symbol_of_uf_cmn_h(lib):
    from paper_2606_09150_b200 import cmn_binding
    hdr = open(os.path.join(ROOT, "include", "uf_cmn.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(uf_cmn_[a-z_0-9]+)\s*\(", hdr)))
    assert declared == sorted(cmn_binding.CMN_SYMBOLS), (declared, sorted(cmn_binding.CMN_SYMBOLS))
    for name in declared:
        assert hasattr(lib, name), f"libuf.so does not export {name}"
    # no GPU here: creating a network fails loudly (no CPU fallback), unsupported widths are refused first
    with pytest.raises(uf.UFError) as e:
        uf.uf_cmn_create(16, 16, (48,), 1, (1,), (1,), 8, 8, 1)
    assert e.value.code == binding.UF_ERR_UNSUPPORTED
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(uf.UFError) as e:
            uf.uf_cmn_create(16, 16, (64,), 1, (1,), (1,), 8, 8, 1)
        assert e.value.code == binding.UF_ERR_CUDA


def test_library_contains_sm100a_tensor_core_code():
    """The shipped binary holds sm_100a SASS with tcgen05 MMA (UTC*MMA), TMEM loads (LDTM) and TMA."""
    import shutil
    import subprocess
    uf.build()
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([cuobjdump, "-sass", uf.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in sass
    for mnemonic in ("UTCHMMA", "LDTM", "STTM", "UTMALDG", "UTMASTG"):
        assert mnemonic in sass, f"{mnemonic} missing from the SASS"


def _host_ctx(C, S=1, H=2, d=128, B=128, nmax=1000, k_min=4):
    return uf.uf_ctx_create(H, d, B, nmax, C, S, k_min, device=-1)


def test_no_gpu_means_loud_failure_not_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(uf.UFError) as ei:
        uf.uf_ctx_create(2, 128, 128, 1000, 3, 1, 4, device=0)
    assert ei.value.code == binding.UF_ERR_CUDA
    ctx = _host_ctx(3)
    try:
        uf.uf_kv_append(ctx, None, None, 10, 256, 128)
        with pytest.raises(uf.UFError) as ei:
            uf.uf_select_blocks(ctx, None, 10, 256, 128, 1, -1)
        assert ei.value.code == binding.UF_ERR_STATE
        with pytest.raises(uf.UFError) as ei:
            uf.uf_sparse_attn_fwd(ctx, None, None, None, 10, 256, 128)
        assert ei.value.code == binding.UF_ERR_STATE
    finally:
        uf.uf_ctx_destroy(ctx)


def test_config_validation(lib):
    for bad in [dict(H=0), dict(d=96), dict(B=48), dict(C=0), dict(C=17), dict(S=5), dict(nmax=0)]:
        kw = dict(C=3, S=1, H=2, d=128, B=128, nmax=1000)
        kw.update(bad)
        with pytest.raises(uf.UFError) as ei:
            _host_ctx(**kw)
        assert ei.value.code == binding.UF_ERR_INVALID_ARG


@pytest.mark.parametrize("C", [1, 2, 3, 5])
def test_slot_map_matches_oracle_constant_window(lib, C):
    """Closed form slot = c mod C (SURVEY 8(c) pins) and equality with the oracle's state machine."""
    H, d, B, nmax = 1, 32, 32, 100
    ctx = _host_ctx(C, H=H, d=d, B=B, nmax=nmax)
    orc = UFOracle(H, d, B, nmax, C)
    z = np.zeros((nmax, H, d))
    try:
        for c in range(20):
            uf.uf_kv_append(ctx, None, None, nmax, H * d, d)
            slot = orc.kv_append(z, z)
            sm = uf.uf_get_slot_map(ctx, C)
            assert sm == tuple(orc.slot_map())
            assert sm[0][c % C] == c and slot == c % C
            assert sorted(x for x in sm[0] if x >= 0) == list(range(max(0, c - C + 1), c + 1))
    finally:
        uf.uf_ctx_destroy(ctx)


def test_slot_map_matches_oracle_random_windows_and_budget(lib):
    rng = np.random.default_rng(7)
    H, d, B, nmax, C, S = 1, 32, 32, 200, 6, 2
    ctx = _host_ctx(C, S=S, H=H, d=d, B=B, nmax=nmax, k_min=4)
    orc = UFOracle(H, d, B, nmax, C, S, 4)
    try:
        for c in range(60):
            n = int(rng.integers(1, nmax + 1))
            win = int(rng.integers(0, C + 1))
            z = np.zeros((n, H, d))
            uf.uf_kv_append(ctx, None, None, n, H * d, d, win)
            orc.kv_append(z, z, win)
            assert uf.uf_get_slot_map(ctx, C) == tuple(orc.slot_map())
            n_cand = len(orc.candidate_ids())
            for count, pct in [(-1, 25), (-1, 0), (-1, 100), (0, -1), (3, -1), (10_000, -1)]:
                assert uf.uf_query_topk(ctx, count, pct) == (n_cand, orc.topk_budget(n_cand, count, pct))
        uf.uf_ctx_reset(ctx)
        assert uf.uf_get_slot_map(ctx, C) == ([-1] * C, 0, -1)
    finally:
        uf.uf_ctx_destroy(ctx)


def test_append_argument_errors(lib):
    ctx = _host_ctx(3, nmax=100)
    try:
        with pytest.raises(uf.UFError) as ei:
            uf.uf_kv_append(ctx, None, None, 101, 256, 128)
        assert ei.value.code == binding.UF_ERR_CAPACITY
        with pytest.raises(uf.UFError) as ei:
            uf.uf_kv_append(ctx, None, None, 0, 256, 128)
        assert ei.value.code == binding.UF_ERR_INVALID_ARG
        with pytest.raises(uf.UFError) as ei:
            uf.uf_kv_append(ctx, None, None, 10, 256, 128, 4)
        assert ei.value.code == binding.UF_ERR_CAPACITY
        with pytest.raises(uf.UFError) as ei:
            uf.uf_query_topk(ctx, -1, 25)          # nothing appended yet
        assert ei.value.code == binding.UF_ERR_STATE
        assert "uf_" in uf.uf_last_error(ctx) or uf.uf_last_error(ctx) == ""
    finally:
        uf.uf_ctx_destroy(ctx)
