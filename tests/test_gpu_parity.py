"""Parity of the CUDA path (through the C ABI, via the thin binding) against the CPU oracle.

Tolerances are BASELINE.json's: relative Frobenius error <= 1e-11 on the upper triangles of U,
U^-1 and H~; eigenvector residual <= 100; S-orthonormality <= 1e-10.  Inputs: the BASELINE recipe
(workloads.py) at sizes the oracle finishes in seconds, spanning one tile, several tiles and ragged
tails, even and odd N (odd N takes the non-TMA loader).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2502_02460_b200 import metrics as M
from paper_2502_02460_b200 import workloads as wl

pytestmark = pytest.mark.gpu

SIZES = [1, 2, 3, 5, 17, 100, 128, 130, 255, 256, 257, 384, 512, 700]


def _gs():
    from paper_2502_02460_b200 import gs
    return gs


def _dev(a):
    """numpy (any order) -> column-major CUDA tensor"""
    t = torch.from_numpy(np.ascontiguousarray(a))
    return wl.to_colmajor(t.cuda())


def _oracle_all(p, nev):
    H, S = p.H.numpy(), p.S.numpy()
    U = oracle.cholesky(S)
    V = oracle.invert_upper(U)
    Ht = oracle.to_standard(H, V)
    return H, S, U, V, Ht


@pytest.mark.parametrize("N", SIZES)
def test_stages_against_oracle(N):
    gs = _gs()
    p = wl.small_pencil(N, seed=N)
    nev = max(1, (2 * N) // 3)
    H, S, U_o, V_o, Ht_o = _oracle_all(p, nev)
    plan = gs.Plan(N, nev)

    # --- step 1: Cholesky, in place; lower triangle of the input is garbage-filled on purpose:
    # gs_cholesky must read the upper triangle only.
    S_in = np.triu(S) + np.tril(np.full((N, N), 123.0), -1)
    U_g = _dev(S_in)
    plan.cholesky(U_g)
    assert plan.last_info() == 0
    assert M.rel_frob_upper(U_g.cpu(), U_o) <= M.TOL_FROB
    assert M.strictly_lower_max(U_g.cpu()) == 0.0

    # --- step 2: inversion, fed with the ORACLE's U (garbage below the diagonal: only the upper
    # triangle may be read) so that the stage is judged on its own
    U_dirty = U_o + np.tril(np.full((N, N), -7.0), -1)
    V_g = wl.colmajor_empty(N, N, device="cuda")
    V_g.fill_(99.0)
    plan.invert_triangular(_dev(U_dirty), V_g)
    assert plan.last_info() == 0
    assert M.rel_frob_upper(V_g.cpu(), V_o) <= M.TOL_FROB
    assert M.strictly_lower_max(V_g.cpu()) == 0.0

    # --- step 3: two-sided transform, fed with the oracle's V (dirty lower triangle)
    V_dirty = V_o + np.tril(np.full((N, N), 5.0), -1)
    Ht_g = wl.colmajor_empty(N, N, device="cuda")
    Ht_g.fill_(-3.0)
    plan.to_standard(_dev(H), _dev(V_dirty), Ht_g)
    assert plan.last_info() == 0
    assert M.rel_frob_upper(Ht_g.cpu(), Ht_o) <= M.TOL_FROB
    if N > 1:   # strictly-lower part of the output buffer is left untouched
        low = torch.tril(Ht_g.cpu(), -1)
        assert torch.all(low[torch.tril(torch.ones(N, N, dtype=torch.bool), -1)] == -3.0)

    # --- back-transform on an identical dense C~ (reading Q8), rectangular, ragged nev
    Ct = wl.dense_rhs(N, nev, seed=N)
    C_o = oracle.backtransform(V_o, Ct.numpy())
    C_g = wl.colmajor_empty(N, nev, device="cuda")
    plan.backtransform(_dev(V_dirty), Ct.cuda().t().contiguous().t(), C_g)
    assert plan.last_info() == 0
    assert M.rel_frob(C_g.cpu(), C_o) <= M.TOL_FROB
    plan.close()


@pytest.mark.parametrize("N", [64, 256, 700, 1024])
def test_chained_path_against_oracle(N):
    """The four calls chained on the GPU's own intermediates, as a user runs them."""
    gs = _gs()
    p = wl.small_pencil(N, seed=1000 + N)
    H, S, U_o, V_o, Ht_o = _oracle_all(p, N)
    plan, U, Uinv, Ht = gs.generalized_to_standard(p.H.cuda().t().contiguous().t(), p.S.cuda().t().contiguous().t())
    assert M.rel_frob_upper(U.cpu(), U_o) <= M.TOL_FROB
    assert M.rel_frob_upper(Uinv.cpu(), V_o) <= M.TOL_FROB
    assert M.rel_frob_upper(Ht.cpu(), Ht_o) <= M.TOL_FROB
    plan.close()


def test_config0_end_to_end():
    """BASELINE config 0 exactly: the three acceptance metrics, with the eigensolve (off the hot
    path) done by the oracle's Jacobi on the GPU's H~."""
    gs = _gs()
    cfg = wl.CONFIGS[0]
    p = wl.make_config(0)
    H, S = p.H.numpy(), p.S.numpy()
    ref = oracle.generalized_eigh(H, S, cfg.nev)
    plan, U, Uinv, Ht = gs.generalized_to_standard(_dev(H), _dev(S), cfg.nev)
    assert M.rel_frob_upper(U.cpu(), ref["U"]) <= M.TOL_FROB
    assert M.rel_frob_upper(Uinv.cpu(), ref["V"]) <= M.TOL_FROB
    assert M.rel_frob_upper(Ht.cpu(), ref["Ht"]) <= M.TOL_FROB
    eps, Q, _ = oracle.jacobi(oracle.hermitian_from_upper(Ht.cpu().numpy()))
    Ct = np.asfortranarray(Q[:, :cfg.nev])
    C = wl.colmajor_empty(cfg.N, cfg.nev, device="cuda")
    plan.backtransform(Uinv, _dev(Ct), C)
    plan.last_info()
    Cn = C.cpu().numpy()
    assert M.eig_residual(H, S, Cn, eps[:cfg.nev]) <= M.TOL_RESIDUAL
    assert M.s_orthonormality(S, Cn) <= M.TOL_SORTH
    np.testing.assert_allclose(eps[:cfg.nev], ref["eps"], rtol=0, atol=1e-9 * np.abs(ref["eps"]).max())
    plan.close()


def test_not_positive_definite_and_noop_after_failure():
    gs = _gs()
    N = 300
    p = wl.small_pencil(N, seed=3)
    S = p.S.numpy().copy()
    S[200, 200] = -1.0        # first non-positive pivot is 201 (1-based)
    plan = gs.Plan(N, N)
    U = _dev(S)
    plan.cholesky(U)
    with pytest.raises(gs.GsError) as e:
        plan.last_info()
    assert e.value.status == 2 and e.value.info == 201
    # later stages are no-ops while the flag is set
    V = wl.colmajor_empty(N, N, device="cuda")
    V.fill_(42.0)
    plan.invert_triangular(U, V)
    assert plan.last_info(raise_on_failure=False) == 201
    assert torch.all(V == 42.0)
    # a fresh gs_cholesky clears the flag
    U2 = _dev(p.S.numpy())
    plan.cholesky(U2)
    assert plan.last_info() == 0
    # NaN is caught as well
    S = p.S.numpy().copy()
    S[10, 10] = np.nan
    plan.cholesky(_dev(S))
    assert plan.last_info(raise_on_failure=False) == 11
    plan.close()


def test_argument_errors():
    gs = _gs()
    with pytest.raises(gs.GsError):
        gs.Plan(0)
    with pytest.raises(gs.GsError):
        gs.Plan(8, nev=9)
    plan = gs.Plan(64, 0)
    S = wl.colmajor_empty(64, 64, device="cuda")
    with pytest.raises(gs.GsError) as e:
        plan.invert_triangular(S, S)        # aliasing
    assert e.value.status == 1
    with pytest.raises(ValueError):
        plan.cholesky(torch.empty((64, 64), dtype=torch.float64, device="cuda"))   # row-major
    plan.backtransform(None, None, None)    # nev == 0: no-op
    plan.close()


@pytest.mark.parametrize("N,cplx", [(300, False), (2500, False), (1100, True)])
def test_host_buffer_entry_points_match_the_device_path(N, cplx):
    """gs_reduce_host / gs_backtransform_host (pinned host buffers, copies inside) give bit for bit what
    the device-pointer calls give: same kernels, same order.  N = 2500 spans five 512-column H2D chunks."""
    gs = _gs()
    nev = N // 3 if N != 2500 else 2200      # 2200 columns: the back-transform runs in six column chunks
    dt = torch.complex128 if cplx else torch.float64
    p = wl.small_pencil(N, seed=77, complex=cplx, device="cuda")
    plan, U, V, Ht = gs.generalized_to_standard(p.H, p.S, nev)
    Ct = wl.dense_rhs(N, nev, seed=5, complex=cplx, device="cuda")
    C = wl.colmajor_empty(N, nev, dtype=dt, device="cuda")
    plan.backtransform(V, Ct, C)
    plan.last_info()

    def host(rows, cols, src=None):
        h = torch.empty((cols, rows), dtype=dt).pin_memory()      # column-major image of a rows x cols matrix
        if src is not None:
            h.copy_(src.t())
        return h

    hH, hS, hCt = host(N, N, p.H), host(N, N, p.S), host(N, nev, Ct)
    hU, hV, hHt, hC = host(N, N), host(N, N), host(N, N), host(N, nev)
    hHt.fill_(-9.0)
    # only the upper triangle of S and the lower triangle of H cross the link: the other triangles of the
    # host buffers and whatever the scratch held before must never be read (NaN would spread)
    nan = float("nan")
    hS.t()[torch.tril(torch.ones(N, N, dtype=torch.bool), -1)] = nan
    hH.t()[torch.triu(torch.ones(N, N, dtype=torch.bool), 1)] = nan
    scratch = torch.full((plan.host_scratch_bytes(),), 0xFF, dtype=torch.uint8, device="cuda")   # all-ones bytes = NaN
    plan.reduce_host(hH, hS, hU, hV, hHt, scratch)
    plan.backtransform_host(hCt, hC, scratch)
    assert torch.equal(torch.triu(hU.t()), torch.triu(U.cpu()))
    assert torch.equal(torch.triu(hV.t()), torch.triu(V.cpu()))
    assert torch.equal(torch.triu(hHt.t()), torch.triu(Ht.cpu()))
    assert torch.equal(hC.t(), C.cpu())
    assert torch.count_nonzero(torch.tril(hU.t(), -1)) == 0 and torch.count_nonzero(torch.tril(hV.t(), -1)) == 0
    esz = 16 if cplx else 8
    assert 0 < plan.reduce_host_d2h_bytes() <= N * N * esz
    assert N * (N + 1) * esz <= plan.reduce_host_h2d_bytes() <= (N * N + 512 * N) * esz
    plan.close()
