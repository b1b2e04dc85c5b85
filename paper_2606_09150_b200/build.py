"""Build libuf.so (the C-ABI library of include/uf.h) in-tree with nvcc for sm_100a.

    python -m paper_2606_09150_b200.build [--force]

nvcc cross-compiles without a GPU.  The library links the CUDA runtime statically and resolves
the one driver entry point it needs (cuTensorMapEncodeTiled) at run time, so it loads on a box
without libcuda (the CPU test box) and fails loudly, with UF_ERR_CUDA, at uf_ctx_create there.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG_DIR)
CSRC = os.path.join(PKG_DIR, "csrc")
LIB = os.path.join(PKG_DIR, "libuf.so")

SOURCES = ["uf_api.cu", "uf_append.cu", "uf_fused_append.cu", "uf_select.cu", "uf_attn_generic.cu", "uf_attn_sm100.cu",
           "uf_cmn.cu", "uf_select_static.cu"]
HEADERS = [os.path.join(CSRC, "uf_internal.h"), os.path.join(CSRC, "uf_sm100_ptx.h"), os.path.join(ROOT, "include", "uf.h"),
           os.path.join(ROOT, "include", "uf_cmn.h"), os.path.join(ROOT, "include", "uf_static.h")]

NVCC_FLAGS = [
    "-O3", "-std=c++17",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo",
    "-Xcompiler", "-fPIC",
    "-shared",
    "-cudart", "static",
]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA extension cannot be built")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every .cu of the package into libuf.so; returns its path."""
    if not force and not is_stale():
        return LIB
    cmd = [_nvcc(), *NVCC_FLAGS, "-I", os.path.join(ROOT, "include"), "-I", CSRC, "-o", LIB]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES]
    proc = subprocess.run(cmd, capture_output=True, text=True)
    if proc.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + proc.stdout + proc.stderr)
    if verbose:
        sys.stderr.write(proc.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
