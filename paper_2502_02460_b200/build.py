"""Build the CUDA libraries in-tree with nvcc for sm_100a.

    python -m paper_2502_02460_b200.build [--force]

Produces paper_2502_02460_b200/libgs.so (the product: C ABI of include/gs.h) and
paper_2502_02460_b200/libgs_peak.so (FP64 peak microbenchmark used by bench.py for the roofline
denominator).  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
NVCC_FLAGS = [
    "-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "shared",
]
TARGETS = {
    "libgs.so": ["gs.cu"],
    "libgs_peak.so": ["fp64_peak.cu"],
}


def _sources_mtime() -> float:
    m = 0.0
    for root in (CSRC, os.path.join(os.path.dirname(HERE), "include")):
        for f in os.listdir(root):
            if f.endswith((".cu", ".cuh", ".h")):
                m = max(m, os.path.getmtime(os.path.join(root, f)))
    return m


# a diagnostic build of libgs.so with per-CTA time stamps in the tridiagonalisation's step kernels (trace_tridiag.py);
# built only on request, never loaded by gs.py
TRACE_TARGET = ("libgs_trace.so", ["gs.cu"], ["-DGS_SV_TRACE"])


def build(force: bool = False, verbose: bool = False, trace: bool = False) -> list[str]:
    nvcc = os.environ.get("NVCC", "nvcc")
    out = []
    newest = _sources_mtime()
    targets = [(lib, srcs, []) for lib, srcs in TARGETS.items()] + ([TRACE_TARGET] if trace else [])
    for lib, srcs, defines in targets:
        path = os.path.join(HERE, lib)
        out.append(path)
        if not force and os.path.exists(path) and os.path.getmtime(path) >= newest:
            continue
        cmd = [nvcc] + NVCC_FLAGS + defines + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", path] + [os.path.join(CSRC, s) for s in srcs]
        subprocess.run(cmd, check=True)
    return out


if __name__ == "__main__":
    for p in build(force="--force" in sys.argv, verbose="-v" in sys.argv, trace="--trace" in sys.argv):
        print(p)
