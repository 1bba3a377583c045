"""Parity of gs_density_matrix (NEXT-1: P_ij = sum_l f_l c*_li c_lj) against the oracle."""
import numpy as np
import pytest
import torch

import oracle
from paper_2502_02460_b200 import metrics as M
from paper_2502_02460_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _dev(a):
    return wl.to_colmajor(torch.from_numpy(np.ascontiguousarray(a)).cuda())


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nev", [(1, 1), (5, 3), (17, 17), (100, 37), (129, 64), (256, 255), (257, 100), (700, 333)])
def test_density_matrix_against_oracle(N, nev, cplx):
    from paper_2502_02460_b200 import gs
    dt = torch.complex128 if cplx else torch.float64
    C = wl.dense_rhs(N, nev, seed=N + nev, complex=cplx)
    rng = np.random.default_rng(N * 1000 + nev)
    f = rng.uniform(0.0, 2.0, nev)
    f[0] = 0.0                                            # an empty state contributes nothing
    P_o = oracle.density_matrix(C.numpy(), f)
    plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
    P = wl.colmajor_empty(N, N, dtype=dt, device="cuda")
    P.fill_(-3.0)
    plan.density_matrix(wl.to_colmajor(C.cuda()), torch.from_numpy(f).cuda(), P)
    assert plan.last_info() == 0
    assert M.rel_frob_upper(P.cpu(), P_o) <= M.TOL_FROB
    if cplx:
        assert torch.all(torch.diagonal(P).imag == 0)
    if N > 1:
        low = P.cpu()[torch.tril(torch.ones(N, N, dtype=torch.bool), -1)]
        assert torch.all(low == -3.0)                      # strictly-lower part untouched
    plan.close()


def test_density_matrix_of_the_path_counts_electrons():
    """End of the chain at config 1's size: C from the GPU path (off-path eigh in between), then
    sum_ij P_ij S_ij = sum_l f_l (Eqs. 3-4) and parity on a leading block."""
    from paper_2502_02460_b200 import gs
    cfg = wl.CONFIGS[1]
    N, nev = cfg.N, cfg.nev
    p = wl.make_pencil(N, cfg.box, cfg.seed, device="cuda")
    plan, U, V, Ht = gs.generalized_to_standard(p.H, p.S, nev)
    eps, Q = torch.linalg.eigh(torch.triu(Ht) + torch.triu(Ht, 1).t())
    C = wl.colmajor_empty(N, nev, device="cuda")
    plan.backtransform(V, wl.to_colmajor(Q[:, :nev].contiguous()), C)
    f = torch.full((nev,), 2.0, dtype=torch.float64, device="cuda")
    P = wl.colmajor_zeros(N, N, device="cuda")
    plan.density_matrix(C, f, P)
    assert plan.last_info() == 0
    Pf = torch.triu(P) + torch.triu(P, 1).t()
    assert abs((Pf * p.S).sum().item() - 2.0 * nev) <= 1e-8 * 2.0 * nev
    k = 512
    P_o = oracle.density_matrix(C[:k, :].cpu().numpy(), f.cpu().numpy())     # leading rows nest
    assert M.rel_frob_upper(P[:k, :k].cpu(), P_o) <= M.TOL_FROB
    plan.close()


def test_density_matrix_nev_zero_writes_zeros():
    from paper_2502_02460_b200 import gs
    plan = gs.Plan(200, 0)
    P = wl.colmajor_empty(200, 200, device="cuda")
    P.fill_(7.0)
    plan.density_matrix(None, None, P)
    assert plan.last_info() == 0
    assert torch.all(torch.triu(P) == 0) and torch.all(torch.tril(P, -1)[torch.tril(torch.ones(200, 200, dtype=torch.bool, device="cuda"), -1)] == 7.0)
    plan.close()
