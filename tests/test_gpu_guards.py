"""Out-of-bounds WRITE detection with guard zones (the stand-in for `compute-sanitizer --tool memcheck`, which
this GPU pool refuses to run -- profiles/r02_sanitizer.md): every buffer a call may write, and the plan's
workspace, is carved out of ONE arena between 64 KiB guard zones filled with a sentinel; after every entry
point of include/gs.h has run at ragged sizes (N = 100, 257, 300: partial tiles, partial leaf blocks, odd N ->
non-TMA loader) the guard zones must be untouched, byte for byte.  Inputs are carved the same way, so a store
through a wrong pointer cannot hide in an input either: inputs are compared with their pristine copies.
Reads out of bounds cannot be seen this way; they are covered by NaN-poisoning what a call must not read
(tests/test_gpu_parity.py, tests/test_gpu_sharded.py) and by TMA's own bounds handling.
"""
import numpy as np
import pytest
import torch

from paper_2502_02460_b200 import workloads as wl

pytestmark = pytest.mark.gpu

GUARD = 64 * 1024
SENTINEL = 0xA5


class Arena:
    def __init__(self, nbytes: int):
        self.buf = torch.full((nbytes,), SENTINEL, dtype=torch.uint8, device="cuda")
        self.off = GUARD
        self.guards = []          # (start, end) byte ranges that must stay SENTINEL
        self.last_end = 0

    def take(self, nbytes: int) -> torch.Tensor:
        start = (self.off + 255) // 256 * 256
        base = self.buf.data_ptr()
        start += (-(base + start)) % 256            # 256-byte aligned device address
        self.guards.append((self.last_end, start))
        self.off = start + nbytes + GUARD
        self.last_end = start + nbytes
        assert self.off <= self.buf.numel()
        return self.buf[start:start + nbytes]

    def matrix(self, rows: int, cols: int, dtype) -> torch.Tensor:
        es = 16 if dtype == torch.complex128 else 8
        raw = self.take(rows * cols * es)
        return raw.view(dtype).view(cols, rows).t()      # column-major, ld = rows

    def check(self):
        self.guards.append((self.last_end, self.buf.numel()))
        for a, b in self.guards:
            seg = self.buf[a:b]
            assert bool((seg == SENTINEL).all()), f"guard zone [{a}, {b}) was written"
        self.guards.pop()


@pytest.mark.parametrize("N,cplx", [(100, False), (257, False), (300, False), (100, True), (257, True)])
def test_no_call_writes_outside_its_buffers(N, cplx):
    from paper_2502_02460_b200 import gs, sharded
    dt = torch.complex128 if cplx else torch.float64
    es = 16 if cplx else 8
    nev = max(2, (2 * N) // 3) & ~1
    p = wl.small_pencil(N, seed=N + 5, complex=cplx, device="cuda")
    plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
    L = gs.lib()
    ws_bytes = plan.workspace.numel()
    arena = Arena(22 * (N * N * es + 2 * GUARD) + ws_bytes + plan.evp_workspace_bytes() + 8 * GUARD)
    ws = arena.take(ws_bytes)
    assert L.gs_plan_set_workspace(plan._h, ws.data_ptr(), ws_bytes) == 0
    H, S, U, V, Ht, G, Vw, Vx, Htx, P = (arena.matrix(N, N, dt) for _ in range(10))
    Ct, C = arena.matrix(N, nev, dt), arena.matrix(N, nev, dt)
    f = arena.take(nev * 8).view(torch.float64)
    H.copy_(p.H)
    S.copy_(p.S)
    Ct.copy_(wl.dense_rhs(N, nev, seed=2, complex=cplx, device="cuda"))
    f.copy_(torch.linspace(2.0, 0.0, nev, dtype=torch.float64, device="cuda"))
    H0, S0, Ct0 = H.clone(), S.clone(), Ct.clone()

    U.copy_(S)
    plan.cholesky(U)
    plan.invert_triangular(U, V)
    plan.to_standard(H, V, Ht)
    plan.backtransform(V, Ct, C)
    plan.density_matrix(C, f, P)
    assert plan.last_info() == 0
    # column-range forms with a push target
    Vx.zero_()
    plan.set_push_targets(gs.GS_PUSH_UINV, [Vx.data_ptr()])
    for c0, c1 in sharded.column_ranges(N, 2, plan.block):
        if c1 > c0:
            U.copy_(S)
            plan.cholesky_leading(U, c1)
            plan.invert_triangular_cols(U, Vw, c0, c1 - c0)
            plan.to_standard_g_cols(H, Vw, G, c0, c1 - c0)
    for c0, c1 in sharded.column_ranges(N, 2, plan.block):
        if c1 > c0:
            plan.to_standard_cols(Vx, G, Htx, c0, c1 - c0)
    plan.backtransform_cols(V, Ct, C, 0, nev)
    assert plan.last_info() == 0
    plan.set_push_targets(gs.GS_PUSH_UINV, [])
    # step 1 in its sharded form: two emulated ranks on this one stream would wait for each other, so one rank here (the
    # same launches minus the copies; tests/test_gpu_sharded_chol.py runs the ranks), and the allocation-free density matrix
    Us = arena.matrix(N, N, dt)
    Us.copy_(S)
    plan.cholesky_sharded(Us, 0, 1)
    Ps = arena.matrix(N, N, dt)
    Ps.copy_(P)
    plan.density_matrix_static(C, f, Ps)
    assert plan.last_info() == 0
    assert torch.equal(torch.triu(Ps), torch.triu(P))
    assert ((torch.triu(Us) - torch.triu(U)).norm() / torch.triu(U).norm()).item() < 1e-13
    # the standard eigensolver (NEXT-4), when the library has it
    if hasattr(plan, "standard_eigh"):
        A = arena.matrix(N, N, dt)
        A.copy_(Ht)
        eps = arena.take(N * 8).view(torch.float64)
        Q = arena.matrix(N, nev, dt)
        plan.standard_eigh(A, eps=eps[:nev], out=Q, workspace_alloc=arena.take)
        assert plan.last_info() == 0
    torch.cuda.synchronize()
    arena.check()
    assert torch.equal(H, H0) and torch.equal(S, S0) and torch.equal(Ct, Ct0)
    # and the results are the right ones (a write that lands inside the right buffer but at the wrong place)
    Ut = torch.triu(U)
    assert ((Ut.conj().t() @ Ut - S0).norm() / S0.norm()).item() < 1e-13
    assert ((Ut @ V - torch.eye(N, dtype=dt, device="cuda")).norm() / N ** 0.5).item() < 1e-11
    assert ((torch.triu(Htx) - torch.triu(Ht)).norm() / torch.triu(Ht).norm()).item() < 1e-11
    plan.close()
