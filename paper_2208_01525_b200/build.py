"""Build libu1u1.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2208_01525_b200.build [--force] [--verbose]

U1U1_NVCC_EXTRA (environment): extra nvcc flags, e.g. "-DTB_TY=8" for the 32 x 8-tile version of the two-step kernel.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libu1u1.so")
SOURCES = ["api.cu", "tma_maps.cu", "step_ref.cu", "step_tiled.cu", "step_tb.cu", "diag_fused.cu", "diag.cu", "gauss_static.cu", "segments.cu", "init.cu"]
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "--shared", "-cudart", "static"]


def _deps():
    out = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    out.append(os.path.join(os.path.dirname(HERE), "include", "u1u1.h"))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in _deps()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("U1U1_NVCC_EXTRA", "").split()
    cmd = [nvcc] + FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
