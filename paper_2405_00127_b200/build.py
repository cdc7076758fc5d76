"""Build libstroke_expand.so (the C-ABI library of include/stroke_expand.h) in-tree with nvcc for sm_100a.

    python -m paper_2405_00127_b200.build [--force]

-fmad=false is deliberate (csrc/sx_math.cuh: the count and write kernels must agree bit for bit, and the
integer-deciding arithmetic follows the paper's fp32 formulas operation by operation); fused multiply-adds in
the vertex evaluation are explicit fmaf().  No --use_fast_math.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libstroke_expand.so")
SOURCES = [os.path.join(CSRC, "sx_kernels.cu"), os.path.join(CSRC, "sx_refined.cu"),
           os.path.join(CSRC, "sx_dash.cu"),
           os.path.join(CSRC, "sx_static.cu")]   # (the second: the kernels of SX_MODE_LINE_REFINED; the third: dashing; the fourth: sx_bin_lines_static)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-fmad=false",
              "-Xcompiler", "-fPIC,-ffp-contract=off", "-shared"]


def _deps():
    out = list(SOURCES)
    for f in os.listdir(CSRC):
        if f.endswith((".cuh", ".h")):
            out.append(os.path.join(CSRC, f))
    out.append(os.path.join(HERE, "..", "include", "stroke_expand.h"))
    return out


def build(force=False, verbose=False):
    if not force and os.path.exists(SO) and all(os.path.getmtime(SO) >= os.path.getmtime(d) for d in _deps()):
        return SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", SO] + SOURCES
    subprocess.check_call(cmd)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
