"""Build libgwstream.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2108_12430_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the
repository snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libgwstream.so")
SOURCES = ["gw_engine.cu", "gw_kernels.cu", "gw_conv_gemm.cu", "gw_bbh_fused.cu", "gw_noalloc.cu"]
HEADERS = ["gw_common.cuh", "gw_ptx.cuh", os.path.join("..", "..", "include", "gwstream.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "--shared"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    trace = ["-DGW_TRACE"] if os.environ.get("GW_TRACE") == "1" else []   # diagnostic build: per-role wait counters
    if os.environ.get("GW_BF16_APPROX_TANH") == "1":                      # experiment: one-MUFU tanh for bf16 as well
        trace.append("-DGW_BF16_APPROX_TANH")
    cmd = [nvcc] + NVCC_FLAGS + trace + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libgwstream.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
