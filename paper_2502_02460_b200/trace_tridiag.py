"""Timeline of one column of the tridiagonalisation (csrc/evp_tridiag.cuh, "Timeline of one column").

    python -m paper_2502_02460_b200.trace_tridiag [--complex] N m [m ...]

Builds the diagnostic library libgs_trace.so (libgs.so compiled with -DGS_SV_TRACE: %globaltimer stamps in the step
kernels S = symv_tma_kernel and C = combine_kernel), runs gs_evp_tridiagonalize on a random symmetric N x N matrix and
prints, for the active blocks of order m and m - 1, when the CTAs of S entered, saw their grid dependency resolved,
streamed and ended, and when C ran -- all in microseconds from the first entry of that S launch.  A measuring aid only:
nothing else loads that library, and its timings include the (small) cost of the stamps.
"""
from __future__ import annotations

import ctypes
import sys

import numpy as np
import torch

from . import build as _build
from . import gs
from . import workloads as wl

TRACE_CTAS = 600


def main(argv=None) -> int:
    argv = sys.argv[1:] if argv is None else list(argv)
    cplx = "--complex" in argv
    argv = [a for a in argv if a != "--complex"]
    if len(argv) < 2:
        print(__doc__, file=sys.stderr)
        return 2
    N, ms = int(argv[0]), [int(x) for x in argv[1:]]
    if not torch.cuda.is_available():
        print("trace_tridiag: no CUDA device", file=sys.stderr)
        return 2
    gs.LIB_PATH = [p for p in _build.build(trace=True) if p.endswith("libgs_trace.so")][0]     # before the first gs.lib()
    L = gs.lib()
    L.gs_trace_tridiag_arm.argtypes = [ctypes.c_int]
    L.gs_trace_tridiag_read.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
    hbm = gs.measured_hbm_gbs() if hasattr(gs, "measured_hbm_gbs") else None
    plan = gs.Plan(N, max(N // 4, 1), dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
    g = torch.Generator(device="cpu")
    g.manual_seed(1)
    A0 = torch.randn(N, N, dtype=torch.complex128 if cplx else torch.float64, generator=g)
    A0 = wl.to_colmajor((A0 + A0.conj().t()).cuda())
    es = 16 if cplx else 8
    A = A0.clone()
    plan.evp_tridiagonalize(A)                       # warm-up: modules loaded, attributes set
    torch.cuda.synchronize()
    for m in ms:
        A.copy_(A0)
        assert L.gs_trace_tridiag_arm(m) == 0
        plan.evp_tridiagonalize(A)
        sv = np.zeros((2, TRACE_CTAS, 8), dtype=np.uint64)
        cc = np.zeros((2, 4), dtype=np.uint64)
        assert L.gs_trace_tridiag_read(sv.ctypes.data, cc.ctypes.data) == 0
        sv, cc = sv.astype(np.int64), cc.astype(np.int64)
        starts = []
        for slot in (0, 1):
            s = sv[slot][sv[slot][:, 1] > 0]
            if len(s) == 0:
                print(f"m={m - slot}: no S launch of that order went through symv_tma_kernel")
                continue
            dots, st = s[s[:, 7] == 1], s[s[:, 7] == 0]
            base = s[:, 0].min()
            us = lambda x: (x - base) / 1e3
            starts.append(s[:, 1].min())
            q = lambda a, f: us(np.percentile(a, f))
            bytes_ = 0.5 * es * (m - slot) ** 2
            span = (st[:, 3].max() - st[:, 2].min()) / 1e3
            print(f"m={m - slot}: S {len(st)} streaming + {len(dots)} panel-dot CTAs | dependency resolved at {us(s[:, 1].min()):.1f}"
                  f" | first item at {q(st[:, 2], 50):.1f} (median) | stream end min / median / max {us(st[:, 3].min()):.1f} / {q(st[:, 3], 50):.1f} / {us(st[:, 3].max()):.1f}"
                  f" | {bytes_ / 1e9:.3f} GB in {span:.1f} us = {bytes_ / span / 1e6:.2f} TB/s"
                  f" | panel dots end {us(dots[:, 3].max()) if len(dots) else float('nan'):.1f}"
                  f" | items per CTA {st[:, 4].min()}..{st[:, 4].max()}, tiles {st[:, 5].min()}..{st[:, 5].max()}"
                  f" | C entry {us(cc[slot][0]):.1f}, start {us(cc[slot][1]):.1f}, end {us(cc[slot][2]):.1f}")
        if len(starts) == 2:
            print(f"   period (dependency resolved -> resolved): {(starts[1] - starts[0]) / 1e3:.1f} us;  the triangle's {0.5 * es * m * m / 1e9:.3f} GB at the HBM copy rate"
                  f" ({hbm or 6549:.0f} GB/s): {0.5 * es * m * m / (hbm or 6549) / 1e3:.1f} us")
    plan.close()
    return 0


if __name__ == "__main__":
    sys.exit(main())
