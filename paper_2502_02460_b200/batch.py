"""NEXT-2: many independent mid-size pencils on ONE GPU.

The paper's "trivial parallelism (e.g., for separate k-points or spin channels)":
K pencils of the same order are independent, so each gets its own plan (host object + workspace) and
its own CUDA stream, and the calls of include/gs.h are simply enqueued round-robin.  A single mid-size
problem cannot fill 148 SMs (its factorisation is a chain of small launches); K of them in flight do.
Only stream plumbing lives here -- every arithmetic step still runs in the kernels of libgs.so.
"""
from __future__ import annotations

import torch

from . import gs
from .workloads import colmajor_empty, colmajor_zeros


class Batch:
    def __init__(self, K: int, N: int, nev: int, complex: bool = False, device=None):
        self.K, self.N, self.nev, self.complex = int(K), int(N), int(nev), bool(complex)
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self.tdtype = torch.complex128 if complex else torch.float64
        dt = gs.GS_COMPLEX128 if complex else gs.GS_REAL64
        self.plans = [gs.Plan(N, nev, dtype=dt, device=self.device) for _ in range(self.K)]
        self.streams = [torch.cuda.Stream(device=self.device) for _ in range(self.K)]

    def _fork(self):
        cur = torch.cuda.current_stream(self.device)
        for s in self.streams:
            s.wait_stream(cur)

    def _join(self):
        cur = torch.cuda.current_stream(self.device)
        for s in self.streams:
            cur.wait_stream(s)

    def alloc(self, cols: int | None = None, zeros: bool = False):
        mk = colmajor_zeros if zeros else colmajor_empty
        return [mk(self.N, self.N if cols is None else cols, dtype=self.tdtype, device=self.device) for _ in range(self.K)]

    def reduce(self, H, S, U, Uinv, Ht):
        """Steps 1-3 of PAPER.md:61-67 for every pencil k: U[k] <- chol(S[k]) (S is not modified),
        Uinv[k], Ht[k].  Returns after ENQUEUEING; the current stream waits for all K streams."""
        self._fork()
        # stage by stage, round-robin over the pencils, so that the K latency-bound chains interleave
        for k in range(self.K):
            with torch.cuda.stream(self.streams[k]):
                U[k].copy_(S[k])
                self.plans[k].cholesky(U[k], stream=self.streams[k])
        for k in range(self.K):
            self.plans[k].invert_triangular(U[k], Uinv[k], stream=self.streams[k])
        for k in range(self.K):
            self.plans[k].to_standard(H[k], Uinv[k], Ht[k], stream=self.streams[k])
        self._join()

    def backtransform(self, Uinv, Ct, C):
        self._fork()
        for k in range(self.K):
            self.plans[k].backtransform(Uinv[k], Ct[k], C[k], stream=self.streams[k])
        self._join()

    def last_info(self):
        return [p.last_info(stream=s) for p, s in zip(self.plans, self.streams)]

    def close(self):
        for p in self.plans:
            p.close()
