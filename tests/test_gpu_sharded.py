"""Parity of the column-range (sharded) forms of steps 2, 3 and the back-transformation against the
CPU oracle, through the C ABI.

One GPU stands in for the R ranks ONE AFTER THE OTHER (no kernel waits on another rank): rank r runs its
column-range calls on buffers that are NaN everywhere it has not written, the test copies only the
slab the rank owns into the exchanged matrices, and before step 3 every column to the right of the
rank's range is poisoned again -- so a rank that reads something the exchange would not have given
it produces NaNs, and the assembled U^-1, H~, C must match the oracle to the north_star tolerance.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2502_02460_b200 import metrics as M
from paper_2502_02460_b200 import sharded
from paper_2502_02460_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _gs():
    from paper_2502_02460_b200 import gs
    return gs


def _nan(N, cols, dtype):
    X = wl.colmajor_empty(N, cols, dtype=dtype, device="cuda")
    X.fill_(float("nan"))
    return X


def _run(N, cplx, world, nev, seed):
    gs = _gs()
    p = wl.small_pencil(N, seed=seed, complex=cplx)
    Hn, Sn = p.H.numpy(), p.S.numpy()
    U_o = oracle.cholesky(Sn)
    V_o = oracle.invert_upper(U_o)
    Ht_o = oracle.to_standard(Hn, V_o)
    dt = p.H.dtype
    H, S = wl.to_colmajor(p.H.cuda()), wl.to_colmajor(p.S.cuda())
    plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
    ranges = sharded.column_ranges(N, world, plan.block)
    U = wl.colmajor_empty(N, N, dtype=dt, device="cuda")
    V_all, G_all, Ht_all = _nan(N, N, dt), _nan(N, N, dt), _nan(N, N, dt)
    for c0, c1 in ranges:                      # steps 1-2 of rank r, then its slabs "go out"
        V_r, G_r = _nan(N, N, dt), _nan(N, N, dt)
        U.copy_(S)
        plan.cholesky_leading(U, c1)           # the rank factors only the leading block it needs ...
        plan.last_info()
        if c1 > 0:
            assert M.rel_frob_upper(U[:c1, :c1].cpu(), U_o[:c1, :c1]) <= M.TOL_FROB
        if c1 < N:
            assert torch.equal(torch.triu(U)[:c1, c1:], torch.triu(S)[:c1, c1:])     # ... and leaves the rest as it was
        U[:, c1:] = float("nan")
        plan.invert_triangular_cols(U, V_r, c0, c1 - c0)
        plan.to_standard_g_cols(H, V_r, G_r, c0, c1 - c0)
        plan.last_info()
        V_all[:, c0:c1] = V_r[:, c0:c1]
        G_all[:, c0:c1] = G_r[:, c0:c1]
    assert torch.isfinite(torch.view_as_real(V_all) if cplx else V_all).all()
    assert M.strictly_lower_max(V_all.cpu()) == 0.0
    assert M.rel_frob_upper(V_all.cpu(), V_o) <= M.TOL_FROB
    for c0, c1 in ranges:                      # step 3 of rank r sees the slabs of ranks <= r only
        V_r, G_r, Ht_r = V_all.clone(), G_all.clone(), _nan(N, N, dt)
        V_r[:, c1:] = float("nan")
        G_r[:, c1:] = float("nan")
        plan.to_standard_cols(V_r, G_r, Ht_r, c0, c1 - c0)
        plan.last_info()
        Ht_all[:, c0:c1] = Ht_r[:, c0:c1]
    Ht_up = torch.triu(Ht_all.cpu())
    assert torch.isfinite(torch.view_as_real(Ht_up) if cplx else Ht_up).all()
    assert M.rel_frob_upper(Ht_up, Ht_o) <= M.TOL_FROB
    if cplx:
        assert float(torch.diagonal(Ht_all).imag.abs().max()) == 0.0
    # untouched below the diagonal blocks (the strictly-lower part of H~ is not written)
    if N > 2 * plan.block:
        assert torch.isnan(Ht_all[N - 1, 0].real if cplx else Ht_all[N - 1, 0])
    if nev > 0:
        Ct = wl.dense_rhs(N, nev, seed=seed + 1, complex=cplx)
        Ctd = wl.to_colmajor(Ct.cuda())
        C = _nan(N, nev, dt)
        for k0, k1 in sharded.even_ranges(nev, world, 2):
            plan.backtransform_cols(V_all, Ctd, C, k0, k1 - k0)
        plan.last_info()
        assert M.rel_frob(C.cpu(), oracle.backtransform(V_o, Ct.numpy())) <= M.TOL_FROB
    plan.close()


@pytest.mark.parametrize("N,cplx,world", [
    (1500, False, 3), (2304, False, 4), (1000, False, 8), (129, False, 2), (100, False, 2),
    (900, True, 3), (1411, True, 5),
])
def test_sharded_columns_against_oracle(N, cplx, world):
    _run(N, cplx, world, nev=(2 * N) // 3, seed=N + world)


@pytest.mark.parametrize("log2p", ["0", "1", "2"])
def test_sharded_small_panels(monkeypatch, log2p):
    """Panels of 1, 2, 4 blocks: many back-substitution steps at a size the oracle finishes quickly."""
    monkeypatch.setenv("GS_SHARD_PANEL_LOG2", log2p)
    _run(1333, False, 3, nev=40, seed=int(log2p) + 70)
    _run(701, True, 2, nev=0, seed=int(log2p) + 80)


def test_one_rank_equals_whole_matrix_calls():
    """world = 1: the column-range calls cover everything; same H~ as the whole-matrix calls to rounding."""
    gs = _gs()
    N = 1792
    p = wl.small_pencil(N, seed=5)
    H, S = wl.to_colmajor(p.H.cuda()), wl.to_colmajor(p.S.cuda())
    plan, U, V, Ht = gs.generalized_to_standard(H, S, 0)
    drv = sharded.ShardedReduction(plan, 0, 1)
    res = drv.reduce(H, S)
    assert torch.equal(res.U, U)            # one rank: the leading block is the whole matrix
    assert M.rel_frob_upper(res.Uinv.cpu(), V.cpu()) <= 1e-13
    assert M.rel_frob_upper(res.Htilde.cpu(), Ht.cpu()) <= 1e-13
    plan.close()


def test_column_range_argument_errors():
    gs = _gs()
    N = 512
    plan = gs.Plan(N, 64)
    A, B, C = (wl.colmajor_zeros(N, N, device="cuda") for _ in range(3))
    for bad in ((64, 128), (0, 100), (-128, 128), (384, 256)):
        with pytest.raises(gs.GsError) as e:
            plan.invert_triangular_cols(A, B, *bad)
        assert e.value.status == 1
        with pytest.raises(gs.GsError):
            plan.to_standard_cols(A, B, C, *bad)
    with pytest.raises(gs.GsError):
        plan.invert_triangular_cols(A, A, 0, N)
    Ct = wl.colmajor_zeros(N, 64, device="cuda")
    Co = wl.colmajor_zeros(N, 64, device="cuda")
    with pytest.raises(gs.GsError):
        plan.backtransform_cols(A, Ct, Co, 32, 64)
    plan.invert_triangular_cols(A, B, 0, 0)      # empty range: no-op
    plan.close()


@pytest.mark.parametrize("N,cplx", [(1100, False), (650, True)])
def test_push_targets_receive_exactly_the_slab(N, cplx):
    """Fused exchange, kernel side (gs_plan_set_push_targets): with two further LOCAL buffers registered as
    push targets, every column-range call leaves in each of them bit for bit what it leaves in its own
    output inside the range (upper part), and touches nothing outside."""
    gs = _gs()
    p = wl.small_pencil(N, seed=3, complex=cplx)
    dt = p.H.dtype
    H, S = wl.to_colmajor(p.H.cuda()), wl.to_colmajor(p.S.cuda())
    nev = N // 2
    plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
    U = wl.colmajor_empty(N, N, dtype=dt, device="cuda")
    U.copy_(S)
    plan.cholesky(U)
    c0, c1 = sharded.column_ranges(N, 3, plan.block)[1]
    assert 0 < c0 < c1 < N
    SENT = -7.25

    def targets(cols):
        t = [wl.colmajor_empty(N, cols, dtype=dt, device="cuda") for _ in range(2)]
        for x in t:
            x.fill_(SENT)
        return t

    def check(own, tgts, a, b, upper):
        for x in tgts:
            inside_own, inside = own[:, a:b], x[:, a:b]
            if upper:
                mask = torch.ones(N, N, dtype=torch.bool, device="cuda").triu()[:, a:b]
                assert torch.equal(inside[mask], inside_own[mask])
            else:
                assert torch.equal(inside, inside_own)
            assert bool((x[:, :a] == SENT).all()) and bool((x[:, b:] == SENT).all())

    V = _nan(N, N, dt)
    tv = targets(N)
    plan.set_push_targets(gs.GS_PUSH_UINV, [x.data_ptr() for x in tv])
    plan.invert_triangular_cols(U, V, c0, c1 - c0)
    plan.last_info()
    check(V, tv, c0, c1, upper=True)
    G = _nan(N, N, dt)
    tg = targets(N)
    plan.set_push_targets(gs.GS_PUSH_G, [x.data_ptr() for x in tg])
    plan.to_standard_g_cols(H, V, G, c0, c1 - c0)
    plan.last_info()
    check(G, tg, c0, c1, upper=True)
    # complete V, G by the whole-range call, then step 3 and the back-transform with targets
    plan.set_push_targets(gs.GS_PUSH_UINV, [])
    plan.set_push_targets(gs.GS_PUSH_G, [])
    plan.invert_triangular_cols(U, V, 0, N)
    plan.to_standard_g_cols(H, V, G, 0, N)
    Ht = _nan(N, N, dt)
    th = targets(N)
    plan.set_push_targets(gs.GS_PUSH_HTILDE, [x.data_ptr() for x in th])
    plan.to_standard_cols(V, G, Ht, c0, c1 - c0)
    plan.last_info()
    check(Ht, th, c0, c1, upper=True)
    Ct = wl.to_colmajor(wl.dense_rhs(N, nev, seed=8, complex=cplx).cuda())
    C = _nan(N, nev, dt)
    tc = targets(nev)
    plan.set_push_targets(gs.GS_PUSH_C, [x.data_ptr() for x in tc])
    k0, k1 = sharded.even_ranges(nev, 3, 2)[1]
    plan.backtransform_cols(V, Ct, C, k0, k1 - k0)
    plan.last_info()
    check(C, tc, k0, k1, upper=False)
    with pytest.raises(gs.GsError):
        plan.set_push_targets(gs.GS_PUSH_C, [1] * 9)
    plan.close()


def test_sharded_reduction_reports_a_non_positive_definite_s():
    gs = _gs()
    N = 640
    p = wl.small_pencil(N, seed=4)
    S = p.S.clone()
    S[300, 300] = -1.0
    plan = gs.Plan(N, 0)
    drv = sharded.ShardedReduction(plan, 0, 1)
    with pytest.raises(gs.GsError) as e:
        drv.reduce(wl.to_colmajor(p.H.cuda()), wl.to_colmajor(S.cuda()))
    assert e.value.status == 2 and e.value.info == 301
    plan.close()
