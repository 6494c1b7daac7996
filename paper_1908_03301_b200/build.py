"""Build libpn.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1908_03301_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the repo
snapshot.  No JIT, no torch extension machinery: plain `nvcc -shared`.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpn.so")
SOURCES = ["pn_api.cu", "pn_setup.cu", "pn_outer.cu", "pn_inner.cu", "pn_fused_tma.cu", "pn_resident.cu", "pn_compact.cu", "pn_chain.cu", "pn_wrap.cu", "pn_onchip.cu", "pn_noalloc.cu"]
HEADERS = [os.path.join(CSRC, "pn_internal.cuh"), os.path.join(CSRC, "pn_tma.cuh"), os.path.join(CSRC, "pn_chain.cuh"), os.path.join(HERE, "..", "include", "pn.h")]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if sources are newer than the library; return the library path."""
    if not force and not _stale():
        return LIB
    cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-Xcompiler", "-fPIC", "-shared", "--threads", "4"]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
